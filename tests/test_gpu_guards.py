"""Out-of-bounds WRITE detection without a sanitizer (compute-sanitizer is closed on this GPU pool): every output and
in-place array of every stage call is a view into a larger buffer whose guard bands are pre-filled with a sentinel and
must come back untouched, bit for bit.  Aligned (guard of 64 elements) and unaligned (guard of 61) placements; ragged,
high-particles-per-cell (slice paths), empty-cell and body/reservoir geometries."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_15622_b200 import fpcl
    fpcl.load()
    return fpcl


@pytest.fixture(scope="module")
def wl():
    from paper_2606_15622_b200 import workloads
    return workloads


class Guarded:
    """Tensors carved out of sentinel-filled buffers; check() verifies every guard band."""

    def __init__(self, torch, guard):
        self.torch, self.guard, self.items = torch, guard, []

    def _sentinel(self, dtype):
        return {self.torch.float32: 1.2345e30, self.torch.float64: 1.2345e300, self.torch.int32: 0x5A5A5A5A}[dtype]

    def empty(self, shape, dtype):
        n = int(np.prod(shape))
        big = self.torch.full((n + 2 * self.guard,), self._sentinel(dtype), dtype=dtype, device="cuda")
        self.items.append((big, n))
        return big[self.guard:self.guard + n].view(*shape)

    def like(self, t):
        v = self.empty(tuple(t.shape), t.dtype)
        v.copy_(t)
        return v

    def check(self, what):
        self.torch.cuda.synchronize()
        for big, n in self.items:
            s = self._sentinel(big.dtype)
            lo, hi = big[: self.guard], big[self.guard + n:]
            assert bool((lo == s).all()) and bool((hi == s).all()), "guard band overwritten after " + what


def _cases(wl):
    yield "ragged", wl.ragged(nx=17, ny=9, seed=11, mean_ppc=35.0), {}
    yield "highppc", wl.ragged(nx=3, ny=2, seed=12, mean_ppc=900.0, empty_frac=0.0), {}
    cfg, st, _ = wl.cylinder(nx=40, ny=30, seed=5, target=40_000)
    yield "cylinder", (dict(cfg, dt=float(np.float32(0.4))), st), dict(per_cell_tau=True)


@pytest.mark.parametrize("guard", [64, 61])
def test_no_write_outside_the_arrays(gpu, wl, guard):
    import torch
    for name, (cfg, st), opt in _cases(wl):
        ctx = gpu.Context(cfg)
        G = Guarded(torch, guard)
        d0 = gpu.to_device(st)
        a = {k: G.like(v) for k, v in d0.items()}
        b = {k: G.empty(tuple(v.shape), v.dtype) for k, v in d0.items()}
        ncell = ctx.ncell
        for closure in (0, 1):
            out = dict(mom=G.empty((ncell, 29 if closure == 0 else 13), torch.float64), coef=G.empty((ncell, 9), torch.float32),
                       flags=G.empty((ncell,), torch.int32), cell_start=G.empty((ncell + 1,), torch.int32))
            out["coef"].zero_(); out["flags"].zero_()
            mlp = gpu.Mlp(wl.xavier_mlp(n_scale=1.0 / 40.0, tau=cfg["tau"], bias_scale=0.1)) if closure else None
            kw = {}
            if opt.get("per_cell_tau"):
                kw = dict(tau_mode=1, tau_ref_n=float(np.float32(cfg["tau"] * cfg["ppc_inf"])), tau_cell=G.empty((ncell,), torch.float32))
            for a_k, v in d0.items():
                a[a_k].copy_(v)
            ctx.step(a, b, 3, out, closure=closure, mlp=mlp, **kw)
            G.check("%s fp_step closure %d" % (name, closure))
            # the stage calls on the sorted output
            cs = out["cell_start"]
            tau_c = kw.get("tau_cell")
            for mode, stride in ((1, 29), (0, 13)):
                mom = G.empty((ncell, stride), torch.float64)
                ctx.cell_moments(b["vx"], b["vy"], b["vz"], cs, mode, out=mom)
                G.check("%s fp_cell_moments mode %d" % (name, mode))
                if mode == 1:
                    coef, flags, kap = G.empty((ncell, 9), torch.float32), G.empty((ncell,), torch.int32), G.empty((ncell,), torch.float64)
                    gpu.fp_closure_exact(ctx.h, mom, tau_c, coef, flags, kap)
                    G.check("%s fp_closure_exact" % name)
                    v = [G.like(b[k]) for k in ("vx", "vy", "vz")]
                    ctx.velocity_update(v[0], v[1], v[2], b["pid"], cs, mom, coef, 9, flags, tau_cell=tau_c)
                    G.check("%s fp_velocity_update" % name)
                elif mlp is not None:
                    coef, flags = G.empty((ncell, 9), torch.float32), G.empty((ncell,), torch.int32)
                    coef.zero_()
                    gpu.fp_closure_mlp(ctx.h, mom, 13, tau_c, mlp, 0.5, coef, flags)
                    G.check("%s fp_closure_mlp" % name)
        s2 = {k: G.like(v) for k, v in d0.items()}
        ctx.stream_walls(s2, 5)
        G.check("%s fp_stream_walls" % name)
        ctx.close()
