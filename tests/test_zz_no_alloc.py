"""fp_cell_moments_static (include/fpcl.h): the context-free moment gather that allocates nothing -- its scratch is a
file-scope __device__ array of FP_STATIC_MAX_CELLS x 28 doubles -- against the existing fp_cell_moments on the same
inputs, within the moment tolerance of tests/parity_util.py, on two calls in a row that share the array.  Collected last
on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from parity_util import abs_moments, moment_ratio

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_15622_b200 import fpcl
    fpcl.load()
    return fpcl


def _case(gpu, nx, ny, seed, mean_ppc, drift):
    """Cell-sorted velocities and cell_start on the device (the library's own sort) plus the context that made them."""
    from paper_2606_15622_b200 import workloads as wl
    cfg, st = wl.ragged(nx=nx, ny=ny, seed=seed, mean_ppc=mean_ppc, drift=drift)
    ctx = gpu.Context(cfg)
    srt, cs, _ = ctx.sort_by_cell(gpu.to_device(st), want_perm=False)
    return ctx, srt, cs


def _ratio(got, ref, srt, cs):
    v = [srt[k].cpu().numpy() for k in ("vx", "vy", "vz")]
    ref = ref.cpu().numpy()
    return moment_ratio(got.cpu().numpy(), ref, absmom=abs_moments(v[0], v[1], v[2], cs.cpu().numpy(), ref))


def test_static_moments_match_the_context_path_twice_in_a_row(gpu):
    import torch
    # two different ensembles with the SAME number of cells: accumulators the second call failed to clear would add up
    ctx1, s1, cs1 = _case(gpu, 16, 12, 31, 90.0, 0.0)          # ordinary cells (empty and 1-3 particle cells included)
    ctx2, s2, cs2 = _case(gpu, 12, 16, 32, 700.0, 9.09)        # huge cells and a Mach-10 drift
    ncell = 192
    assert ctx1.ncell == ncell and ctx2.ncell == ncell
    for mode, ncol in ((1, 29), (0, 13)):
        want1 = ctx1.cell_moments(s1["vx"], s1["vy"], s1["vz"], cs1, mode)
        want2 = ctx2.cell_moments(s2["vx"], s2["vy"], s2["vz"], cs2, mode)
        got1 = torch.full((ncell, ncol), float("nan"), dtype=torch.float64, device="cuda")
        got2 = torch.full((ncell, ncol), float("nan"), dtype=torch.float64, device="cuda")
        st1 = torch.full((1,), -1, dtype=torch.int32, device="cuda")
        st2 = torch.full((1,), -1, dtype=torch.int32, device="cuda")
        # first call on the device resolves the scratch address and loads the kernels
        gpu.fp_cell_moments_static(s1["vx"].numel(), s1["vx"], s1["vy"], s1["vz"], cs1, ncell, mode, got1, st1)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        # the two calls in a row, in stream order, nothing in between
        gpu.fp_cell_moments_static(s1["vx"].numel(), s1["vx"], s1["vy"], s1["vz"], cs1, ncell, mode, got1, st1)
        gpu.fp_cell_moments_static(s2["vx"].numel(), s2["vx"], s2["vy"], s2["vz"], cs2, ncell, mode, got2, st2)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] >= free_before, "device memory was allocated by fp_cell_moments_static"
        assert int(st1.item()) == 0 and int(st2.item()) == 0
        r1, r2 = _ratio(got1, want1, s1, cs1), _ratio(got2, want2, s2, cs2)
        print("static vs context moments, mode %d: %.3f %.3f of the 1e-6 tolerance" % (mode, r1, r2))
        assert r1 <= 1.0 and r2 <= 1.0
    ctx1.close()
    ctx2.close()


def test_static_moments_limits_and_bad_cell_start(gpu):
    import torch
    ctx, s, cs = _case(gpu, 8, 6, 33, 40.0, 0.0)
    n, ncell = s["vx"].numel(), ctx.ncell
    mom = torch.full((ncell, 29), 7.0, dtype=torch.float64, device="cuda")
    # beyond the static array: refused with a clear message, nothing launched
    big = gpu.FP_STATIC_MAX_CELLS + 1
    with pytest.raises(gpu.FpclError, match="FP_STATIC_MAX_CELLS"):
        gpu.fp_cell_moments_static(0, s["vx"], s["vy"], s["vz"], torch.zeros(big + 1, dtype=torch.int32, device="cuda"), big, 1,
                                   torch.empty((big, 29), dtype=torch.float64, device="cuda"))
    with pytest.raises(gpu.FpclError, match="16-byte"):
        gpu.fp_cell_moments_static(n - 1, s["vx"][1:], s["vy"][1:], s["vz"][1:], cs, ncell, 1, mom)
    # a cell_start that is not a sorted prefix: records untouched, status word says so
    bad = cs.clone()
    bad[3], bad[4] = cs[4].item() + 5, cs[3].item()
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    gpu.fp_cell_moments_static(n, s["vx"], s["vy"], s["vz"], bad, ncell, 1, mom, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 1
    assert bool((mom == 7.0).all())
    # and the next call is clean again (the status word is part of what a call clears)
    gpu.fp_cell_moments_static(n, s["vx"], s["vy"], s["vz"], cs, ncell, 1, mom, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    want = ctx.cell_moments(s["vx"], s["vy"], s["vz"], cs, 1)
    assert _ratio(mom, want, s, cs) <= 1.0
    # the largest size the array holds, no particles: every record zero
    cs0 = torch.zeros(gpu.FP_STATIC_MAX_CELLS + 1, dtype=torch.int32, device="cuda")
    m0 = torch.full((gpu.FP_STATIC_MAX_CELLS, 13), 1.0, dtype=torch.float64, device="cuda")
    gpu.fp_cell_moments_static(0, None, None, None, cs0, gpu.FP_STATIC_MAX_CELLS, 0, m0)
    torch.cuda.synchronize()
    assert bool((m0 == 0.0).all())
    ctx.close()
