"""SURVEY 8(f) NEXT-4 on one GPU: a cavity cut into slabs of rows, each slab with its own fp_ctx on the same device and
the per-step particle exchange done by device-side slicing (paper_2606_15622_b200/dist.py: exchange_in_process), against
the uncut fp_step run.  The stable partition plus the source-ordered exchange hand every slab exactly the sub-sequence of
the uncut array that it owns, so the union of the slabs must equal the uncut run BIT FOR BIT after any number of steps:
positions, velocities, ids and the cell boundaries (PAPER.md:668 runs replicas only; the cut is this build's extension)."""
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


def _slab_run(gpu, D, cfg, st, bounds, nsteps, closure, mlp):
    import torch
    ns = len(bounds) - 1
    nx = cfg["nx"]
    ctxs = []
    for s in range(ns):
        c = gpu.Context(cfg)
        gpu.fp_set_slab(c.h, bounds[s], bounds[s + 1] - bounds[s])
        gpu.fp_set_reproducible(c.h, True)
        ctxs.append(c)
    # initial ownership by row of the initial positions (global cell-index formula: the library's own sort)
    full = gpu.Context(cfg)
    srt, cs0, _ = full.sort_by_cell(gpu.to_device(st), want_perm=False)
    cs0 = cs0.cpu().numpy()
    own = [{k: srt[k][cs0[bounds[s] * nx]:cs0[bounds[s + 1] * nx]].clone() for k in D.FIELDS} for s in range(ns)]
    full.close()
    outs = None
    for it in range(nsteps):
        parts, starts = [], []
        for s in range(ns):
            n = own[s]["x"].numel()
            ctxs[s].stream_walls(own[s], it)
            p = {k: torch.empty_like(v) for k, v in own[s].items()}
            sstart = torch.empty(ns + 1, dtype=torch.int32, device="cuda")
            gpu.fp_slab_partition(ctxs[s].h, n, own[s], p, bounds, sstart)
            parts.append(p)
            starts.append([int(v) for v in sstart.cpu().tolist()])
            assert starts[-1][0] == 0 and starts[-1][-1] == n
        got = D.exchange_in_process(parts, starts)
        outs = []
        for s in range(ns):
            n = got[s]["x"].numel()
            ncell = nx * (bounds[s + 1] - bounds[s])
            b = {k: torch.empty_like(v) for k, v in got[s].items()}
            o = dict(mom=torch.empty((ncell, 29 if closure == 0 else 13), dtype=torch.float64, device="cuda"),
                     coef=torch.zeros((ncell, 9), dtype=torch.float32, device="cuda"),
                     flags=torch.zeros(ncell, dtype=torch.int32, device="cuda"),
                     cell_start=torch.empty(ncell + 1, dtype=torch.int32, device="cuda"))
            gpu.fp_collide(ctxs[s].h, n, got[s], b, closure, mlp, 1.0, 0, 0.0, None, it, o["mom"], o["coef"], o["flags"],
                           o["cell_start"])
            own[s] = b
            outs.append(o)
    torch.cuda.synchronize()
    for c in ctxs:
        c.close()
    return own, outs


@pytest.mark.parametrize("bounds,closure", [([0, 24, 48], 0), ([0, 7, 30, 48], 0), ([0, 24, 48], 1)])
def test_slabs_equal_the_uncut_run(gpu, bounds, closure):
    import torch
    from paper_2606_15622_b200 import dist as D, workloads as wl
    cfg, st = wl.cavity(n=48, ppc=40, kn=0.5, seed=21)
    cfg = dict(cfg, dt=float(np.float32(0.012)))                     # ~0.6 cell per step: steady traffic across the cuts
    mlp = gpu.Mlp(wl.xavier_mlp(n_scale=1.0 / 40.0, tau=cfg["tau"], bias_scale=0.1)) if closure else None
    nsteps = 10
    # uncut reference
    ctx = gpu.Context(cfg)
    gpu.fp_set_reproducible(ctx.h, True)             # per-cell results independent of the cell's offset in the arrays
    a = gpu.to_device(st)
    b = {k: torch.empty_like(v) for k, v in a.items()}
    out = ctx.alloc_step_outputs(closure)
    # same starting order as the slab run (cell-sorted)
    a, _, _ = ctx.sort_by_cell(a, want_perm=False)
    for it in range(nsteps):
        ctx.step(a, b, it, out, closure=closure, mlp=mlp)
        a, b = b, a
    torch.cuda.synchronize()
    own, outs = _slab_run(gpu, D, cfg, st, bounds, nsteps, closure, mlp)
    for k in D.FIELDS:
        union = torch.cat([own[s][k] for s in range(len(own))])
        assert union.numel() == a[k].numel()
        assert torch.equal(union.view(torch.int32), a[k].view(torch.int32)), k
    # cell boundaries: slab s's cell_start, shifted by the particles of the slabs before it
    off, pieces = 0, []
    for s, o in enumerate(outs):
        cs = o["cell_start"].cpu().numpy().astype(np.int64)
        pieces.append(cs[:-1] + off)
        off += int(cs[-1])
    pieces.append(np.array([off]))
    assert np.array_equal(np.concatenate(pieces), out["cell_start"].cpu().numpy().astype(np.int64))
    # per-cell outputs too
    assert torch.equal(torch.cat([o["mom"] for o in outs]), out["mom"])
    assert torch.equal(torch.cat([o["coef"] for o in outs]), out["coef"])
    assert torch.equal(torch.cat([o["flags"] for o in outs]), out["flags"])
    ctx.close()


def test_partition_is_stable_and_counts_add_up(gpu):
    """fp_slab_partition alone: destinations by the global row formula, input order kept inside each destination."""
    import torch
    from paper_2606_15622_b200 import workloads as wl
    cfg, st = wl.ragged(nx=9, ny=31, seed=5, mean_ppc=20.0)
    bounds = [0, 3, 4, 17, 31]
    ctx = gpu.Context(cfg)
    a = gpu.to_device(st)
    b = {k: torch.empty_like(v) for k, v in a.items()}
    sstart = torch.empty(len(bounds), dtype=torch.int32, device="cuda")
    gpu.fp_slab_partition(ctx.h, a["x"].numel(), a, b, bounds, sstart)
    starts = sstart.cpu().numpy()
    inv_dy = np.float32(1.0) / np.float32(cfg["dy"])
    row = np.clip(np.floor((st["y"] - np.float32(cfg["y0"])) * inv_dy), 0, cfg["ny"] - 1).astype(np.int64)
    dest = np.searchsorted(np.array(bounds), row, side="right") - 1
    order = np.argsort(dest, kind="stable")
    assert np.array_equal(starts, np.concatenate([[0], np.cumsum(np.bincount(dest, minlength=len(bounds) - 1))]))
    for k in ("x", "y", "vx", "vy", "vz"):
        assert np.array_equal(b[k].cpu().numpy().view(np.uint32), st[k][order].view(np.uint32)), k
    assert np.array_equal(b["pid"].cpu().numpy().view(np.uint32), st["pid"][order])
    ctx.close()


@pytest.mark.parametrize("seed,closure,inflow", [(30052, 0, True), (30064, 1, False), (30099, 1, True), (30131, 0, False)])
def test_slabs_of_a_ragged_ensemble(gpu, seed, closure, inflow):
    """Random grids, 3..300 particles per cell with empty and few-particle cells, two to five slabs of unequal heights (some
    a single row), diffuse / periodic / reservoir faces, both closures: the slabs' mean densities select other lane-group
    widths than the uncut run's and their cells sit in other chunks, which reproducible mode must not let through to the
    results.  (An earlier reproducible mode only pinned the visiting order inside a cell: a third of such configurations
    differed in the last bit.)"""
    import torch
    from paper_2606_15622_b200 import dist as D, workloads as wl
    rng = np.random.default_rng(seed)
    nx, ny = int(rng.integers(2, 50)), int(rng.integers(4, 50))
    mean_ppc = float(rng.choice([3, 8, 20, 40, 57, 90, 150, 300]))
    if nx * ny * mean_ppc > 4e5:
        mean_ppc = max(3.0, 4e5 / (nx * ny))
    kx, ky = int(rng.choice([wl.WALL_DIFFUSE, wl.WALL_PERIODIC])), int(rng.choice([wl.WALL_DIFFUSE, wl.WALL_PERIODIC]))
    walls = [(kx, 0.6, 0.0, 0.1, 0.0)] * 2 + [(ky, 0.5, 0.1, 0, 0)] * 2
    if inflow:
        walls = [(wl.WALL_INFLOW, 0.5, float(rng.uniform(0.5, 5.0)), 0.0, 0.0)] * 4
    drift = float(walls[0][2]) if inflow else float(rng.choice([0.0, 0.5, 2.0]))
    cfg, st = wl.ragged(nx=nx, ny=ny, seed=seed, mean_ppc=mean_ppc, empty_frac=0.1, walls=walls, drift=drift)
    cfg = dict(cfg, dt=float(np.float32(rng.uniform(0.01, 0.06))))
    mlp = gpu.Mlp(wl.xavier_mlp(n_scale=1.0 / mean_ppc, tau=cfg["tau"], bias_scale=0.1)) if closure else None
    ns = int(rng.integers(2, min(5, ny) + 1))
    bounds = [0] + sorted(rng.choice(np.arange(1, ny), size=ns - 1, replace=False).tolist()) + [ny]
    nsteps = 4
    ctx = gpu.Context(cfg)
    gpu.fp_set_reproducible(ctx.h, True)
    a = gpu.to_device(st)
    b = {k: torch.empty_like(v) for k, v in a.items()}
    out = ctx.alloc_step_outputs(closure)
    a, _, _ = ctx.sort_by_cell(a, want_perm=False)
    for it in range(nsteps):
        ctx.step(a, b, it, out, closure=closure, mlp=mlp)
        a, b = b, a
    torch.cuda.synchronize()
    own, outs = _slab_run(gpu, D, cfg, st, bounds, nsteps, closure, mlp)
    print("seed %d: %dx%d cells, %.0f ppc, walls %s, closure %d, slabs %s" % (seed, nx, ny, mean_ppc, [w[0] for w in walls], closure, bounds))
    for k in D.FIELDS:
        union = torch.cat([own[s][k] for s in range(len(own))])
        assert torch.equal(union.view(torch.int32), a[k].view(torch.int32)), k
    assert torch.equal(torch.cat([o["mom"] for o in outs]), out["mom"])
    assert torch.equal(torch.cat([o["coef"] for o in outs]), out["coef"])
    ctx.close()
