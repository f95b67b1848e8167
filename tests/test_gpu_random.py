"""Randomised stage-by-stage comparison with the oracle: grids from 1 to ~3000 cells, 3 to 1500 particles per cell (every
lane-group width, the giant-cell and the 512-particle-slice paths), empty / two- / three-particle cells, bulk speeds up to
Mach 30, diffuse / periodic / open / reservoir faces, both conservation modes, eps2 on and off, scalar and per-cell tau.
The seeds below are configurations on which an earlier build of the velocity update (or of the reservoir) missed the
tolerance -- two-particle cells whose energy rescaling cancels, hypersonic few-particle cells whose cubic drift amplifies the
rounding of the bulk velocity, re-emitted particles ten thermal speeds out in giant cells, a borderline accept/reject in the
reservoir -- plus a few that always passed.  Every stage gets the ORACLE's output of the previous stage as its input, so the
strict tolerances of tests/parity_util.py apply (1e-6 moments and velocities, 1e-5 coefficients, integers bit for bit)."""
import os

import numpy as np
import pytest

from parity_util import abs_moments, coef_ratio, moment_ratio, velocity_ratio

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_15622_b200 import fpcl
    fpcl.load()
    return fpcl


def _bits(a):
    return np.ascontiguousarray(a).view(np.uint32)


def _theta(m):
    return (m[:, 4] + m[:, 7] + m[:, 9]) / 3.0


def _random_case(wl, seed):
    """Seeded configuration + ensemble (no method arithmetic: sizes, wall kinds, time step, switches)."""
    rng = np.random.default_rng(seed)
    nx = int(rng.integers(1, 70))
    ny = int(rng.choice([1, int(rng.integers(2, 50))]))
    mean_ppc = float(rng.choice([3, 8, 20, 40, 57, 90, 113, 150, 230, 400, 700, 1500]))
    if nx * ny * mean_ppc > 1.5e6:
        mean_ppc = max(3.0, 1.5e6 / (nx * ny))
    drift = float(rng.choice([0.0, 0.0, 0.5, 3.0, 9.09]))
    kinds = [wl.WALL_DIFFUSE, wl.WALL_PERIODIC, wl.WALL_NONE]

    def pick():
        return (int(rng.choice(kinds)), float(rng.uniform(0.3, 1.0)), float(rng.uniform(-0.3, 0.3)),
                float(rng.uniform(-0.3, 0.3)), float(rng.uniform(-0.3, 0.3)))
    wx, wy = pick(), pick()
    walls = [wx, (wx[0],) + pick()[1:], wy, (wy[0],) + pick()[1:]]
    if rng.random() < 0.15:
        walls = [(wl.WALL_INFLOW, 0.5, float(rng.uniform(0.2, 9.0)), 0.0, 0.0)] * 4
    cfg, st = wl.ragged(nx=nx, ny=ny, seed=seed, mean_ppc=mean_ppc, empty_frac=float(rng.choice([0.0, 0.1, 0.5])), walls=walls,
                        drift=drift)
    cfg = dict(cfg, dt=float(np.float32(rng.uniform(0.005, 0.08))), conserve_mode=int(rng.integers(0, 2)),
               eps2_scale=float(rng.choice([0.0, 1.0, 1.0, 3.0])))
    step = int(rng.integers(0, 1 << 40))
    return rng, cfg, st, step


# seed: what it hit before the fix (N = particles in the worst cell, cm = conserve_mode)
SEEDS = [1028, 1034, 1098, 1287,      # N = 2, cm 1: the energy rescaling is a small difference of its terms (up to 23x the tolerance)
         1030, 1164, 1239,            # hypersonic few-particle cells, giant cells with re-emitted particles at rest (cm 1)
         1076, 1077, 1136, 1204,      # N = 2 .. 6, cm 0: degenerate eps2 ~ 1/(tau theta), cubic term of ~3 thermal speeds
         1241, 5012,                  # 230 ppc with diffuse walls at Mach 13; reservoir faces on 1.2M particles (accept/reject flip)
         30172, 30773, 41721,         # bimodal Mach-9 cells of 2,000+ particles (range floor); at-rest tails in Mach-6 cells (fp64 sums)
         40387, 41783, 102080,        # a 9-particle cell on the slice path; two-particle cells whose energy scale is a small part of its terms
         1000, 1001, 1002, 1003]      # controls


# FPCL_RANDOM_CASES=N adds N fresh seeds (the sweep this file's seeds were found with; ~20 cases per second).  11,000 such
# cases left one miss on the final build: 1.03x in a two-particle cell at Mach 52.
SEEDS += list(range(500000, 500000 + int(os.environ.get("FPCL_RANDOM_CASES", "0"))))


@pytest.mark.parametrize("seed", SEEDS)
def test_random_configuration(gpu, orc, seed):
    import torch
    from paper_2606_15622_b200 import workloads as wl
    rng, cfg, st, step = _random_case(wl, seed)
    ctx = gpu.Context(cfg)
    # a0 + a1
    ref = orc.stream_walls(st, cfg, step)
    d = gpu.to_device(st)
    ctx.stream_walls(d, step)
    got = gpu.to_host(d)
    assert np.array_equal(_bits(got["x"]), _bits(ref["x"])) and np.array_equal(_bits(got["y"]), _bits(ref["y"]))
    hit = (_bits(ref["vx"]) != _bits(st["vx"])) | (_bits(ref["vy"]) != _bits(st["vy"])) | (_bits(ref["vz"]) != _bits(st["vz"]))
    sc = np.sqrt(max(w[1] for w in cfg["walls"]))
    for k in ("vx", "vy", "vz"):
        assert np.array_equal(_bits(got[k])[~hit], _bits(st[k])[~hit])
        if hit.any():
            allowed = 1e-6 * np.maximum(np.abs(ref[k][hit].astype(np.float64)), sc)
            assert (np.abs(got[k][hit].astype(np.float64) - ref[k][hit]) <= allowed).all(), k
    # a2 on the oracle's streamed state
    mid = {k: np.ascontiguousarray(v) for k, v in ref.items()}
    s, cs, perm = orc.sort_by_cell(mid, cfg)
    o, gcs, gperm = ctx.sort_by_cell(gpu.to_device(mid))
    assert np.array_equal(gcs.cpu().numpy(), cs)
    assert np.array_equal(gperm.cpu().numpy().view(np.uint32), perm)
    gs = gpu.to_host(o)
    for k in ("x", "y", "vx", "vy", "vz", "pid"):
        assert np.array_equal(_bits(gs[k]), _bits(s[k])), k
    # a3
    csd = torch.from_numpy(cs).cuda()
    dd = gpu.to_device(s)
    moms = {}
    for mode in (0, 1):
        rm = orc.cell_moments(s["vx"], s["vy"], s["vz"], cs, mode)
        gm = ctx.cell_moments(dd["vx"], dd["vy"], dd["vz"], csd, mode).cpu().numpy()
        assert moment_ratio(gm, rm, absmom=abs_moments(s["vx"], s["vy"], s["vz"], cs, rm)) <= 1.0
        moms[mode] = rm
    # a4
    ncell = cs.shape[0] - 1
    tau = rng.uniform(0.3, 2.0, size=ncell).astype(np.float32) if rng.random() < 0.5 else cfg["tau"]
    tau_d = None if np.ndim(tau) == 0 else torch.from_numpy(tau).cuda()
    coef, flags, kappa = orc.closure_exact(moms[1], tau, cfg["eps2_scale"], cfg["min_count"])
    gc, gf = ctx.closure_exact(torch.from_numpy(moms[1]).cuda(), tau_d)
    gc, gf = gc.cpu().numpy(), gf.cpu().numpy().view(np.uint32)
    hard = orc.FLAG_EMPTY | orc.FLAG_LOWCOUNT | orc.FLAG_SINGULAR
    settled = kappa <= 1e6                                  # near the pivot / kappa decision lines the two sides may differ
    assert np.array_equal((gf & hard)[settled], (flags & hard)[settled])
    good = ((flags & (hard | orc.FLAG_ILLCOND)) == 0) & (kappa < 1e8) & ((gf & hard) == 0)
    assert coef_ratio(gc, coef, tau, _theta(moms[1]), np.maximum(1e-5, 1e-13 * kappa), mask=good) <= 1.0
    # a6 on the oracle's coefficients
    coef32 = coef.astype(np.float32)
    rvx, rvy, rvz, rfl = orc.velocity_update(s["vx"], s["vy"], s["vz"], s["pid"], cs, moms[1], coef32, tau, cfg, step, flags)
    fl = torch.from_numpy(flags.view(np.int32).copy()).cuda()
    ctx.velocity_update(dd["vx"], dd["vy"], dd["vz"], dd["pid"], csd, torch.from_numpy(moms[1]).cuda(),
                        torch.from_numpy(coef32).cuda(), step, fl, tau_cell=tau_d)
    gv = (dd["vx"].cpu().numpy(), dd["vy"].cpu().numpy(), dd["vz"].cpu().numpy())
    assert all(np.isfinite(g).all() for g in gv)
    assert np.array_equal(fl.cpu().numpy().view(np.uint32), rfl)
    r = velocity_ratio(gv, (rvx, rvy, rvz), cs, _theta(moms[1]))
    print("seed %d: %d particles, %d cells, conserve_mode %d: velocities %.3f of 1e-6" % (seed, s["x"].shape[0], ncell,
                                                                                         cfg["conserve_mode"], r))
    assert r <= 1.0
    ctx.close()
