"""Pins for the oracle's velocity update (S5) and streaming/walls (S7).  CPU only."""
import math

import numpy as np
import pytest

from paper_2606_15622_b200 import workloads as wl

LANG = lambda tau: np.float32([-1 / tau, 0, 0, -1 / tau, 0, -1 / tau, 0, 0, 0])  # noqa: E731


def _cell(orc, n, seed, shift=(0.3, -0.2, 0.1)):
    cfg, st, _ = wl.grad13_cells(1, 1, n, seed=seed)
    v = np.stack([st["vx"], st["vy"], st["vz"]], 1) + np.float32(shift)
    cs = np.array([0, n], dtype=np.int32)
    return cfg, v.astype(np.float32), cs, st["pid"]


def test_noise_off_langevin_decay(orc):
    """Langevin coefficients => N = 0, alpha = 1, and Eq. 13 reduces to c* = c e^{-dt/tau} + sqrt(theta(1-e^{-2dt/tau})) xi.
    Subtracting the (separately pinned) normals leaves the exact OU decay."""
    cfg, v, cs, pid = _cell(orc, 64, 1)
    cfg.update(conserve_mode=0, eps2_scale=0.0, dt=float(np.float32(0.17)), seed=77)
    tau = 0.9
    mom = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 0)
    vx, vy, vz, fl = orc.velocity_update(v[:, 0], v[:, 1], v[:, 2], pid, cs, mom, LANG(np.float32(tau))[None, :],
                                         np.float32(tau), cfg, step=5)
    assert fl[0] == 0
    U, theta = mom[0, 1:4], (mom[0, 4] + mom[0, 7] + mom[0, 9]) / 3
    tau32 = float(np.float32(tau))
    a = cfg["dt"] / tau32
    xi = orc.normals(pid, 5, 0, 77)
    new = np.stack([vx, vy, vz], 1).astype(np.float64)
    decay = new - U - math.sqrt(theta * (1 - math.exp(-2 * a))) * xi
    # (C_ii + 1/tau) is not exactly zero because the coefficient is stored in fp32: allow 1e-7 relative slack
    np.testing.assert_allclose(decay, (v.astype(np.float64) - U) * math.exp(-a), atol=3e-7)


def test_eq15_expected_energy(orc):
    """Eq. 15 is the value of alpha^2 for which E_xi <|c*|^2> = 3 theta.  Average over many independent noise draws."""
    cfg, v, cs, pid = _cell(orc, 2000, 2)
    cfg.update(conserve_mode=0, eps2_scale=1.0, dt=float(np.float32(0.3)), seed=5)
    tau = 1.0
    mom = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 1)
    rng = np.random.default_rng(0)
    coef = (LANG(tau) + rng.normal(0, 0.3, 9)).astype(np.float32)[None, :]        # an arbitrary (non-exact) closure
    theta = (mom[0, 4] + mom[0, 7] + mom[0, 9]) / 3
    en = []
    for step in range(60):
        vx, vy, vz, fl = orc.velocity_update(v[:, 0], v[:, 1], v[:, 2], pid, cs, mom, coef, tau, cfg, step)
        assert fl[0] == 0
        c = np.stack([vx, vy, vz], 1).astype(np.float64) - mom[0, 1:4]
        en.append((c ** 2).sum(1).mean())
    se = np.std(en) / math.sqrt(len(en))
    assert abs(np.mean(en) - 3 * theta) < 5 * se + 1e-6
    assert se < 0.01 * 3 * theta


def test_exact_closure_gives_alpha_ge_one_and_mode1_conserves(orc):
    cfg, st, _ = wl.grad13_cells(6, 5, 80, seed=8)
    cs = (np.arange(31) * 80).astype(np.int32)
    mom = orc.cell_moments(st["vx"], st["vy"], st["vz"], cs, 1)
    coef, flags, _ = orc.closure_exact(mom, 1.0, float(cfg["eps2_scale"]))
    cfg.update(conserve_mode=1, seed=3)
    vx, vy, vz, fl = orc.velocity_update(st["vx"], st["vy"], st["vz"], st["pid"], cs, mom, coef.astype(np.float32),
                                         1.0, cfg, step=1, flags=flags)
    assert np.all((fl & orc.FLAG_ALPHA) == 0)
    old = np.stack([st["vx"], st["vy"], st["vz"]], 1).astype(np.float64).reshape(30, 80, 3)
    new = np.stack([vx, vy, vz], 1).astype(np.float64).reshape(30, 80, 3)
    assert np.all(np.isfinite(new))
    # momentum and energy per cell, limited by the fp32 rounding of the stored velocities (~6e-8 per particle)
    np.testing.assert_allclose(new.mean(1), old.mean(1), atol=80 ** -0.5 * 3e-7)
    e_old = ((old - old.mean(1, keepdims=True)) ** 2).sum(2).mean(1)
    e_new = ((new - new.mean(1, keepdims=True)) ** 2).sum(2).mean(1)
    np.testing.assert_allclose(e_new, e_old, rtol=3e-7)
    assert np.abs(new - old).max() > 0.01                                # something actually happened


def test_mode0_momentum_only_in_expectation_and_skips(orc):
    cfg, v, cs, pid = _cell(orc, 500, 4)
    cfg.update(conserve_mode=0, seed=9)
    mom = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 0)
    vx, vy, vz, fl = orc.velocity_update(v[:, 0], v[:, 1], v[:, 2], pid, cs, mom, LANG(1.0)[None, :], 1.0, cfg, 0)
    theta = (mom[0, 4] + mom[0, 7] + mom[0, 9]) / 3
    drift = np.array([vx.mean(), vy.mean(), vz.mean()]) - mom[0, 1:4]
    assert np.all(np.abs(drift) < 5 * math.sqrt(theta / 500))            # noise breaks momentum by O(1/sqrt N)
    assert np.any(np.abs(drift) > 1e-6)
    # cells with N < 2 or theta <= 0 are left untouched and flagged
    v1 = np.float32([[1, 2, 3], [4, 4, 4], [4, 4, 4]])
    cs1 = np.array([0, 1, 3, 3], dtype=np.int32)
    m1 = orc.cell_moments(v1[:, 0], v1[:, 1], v1[:, 2], cs1, 0)
    a, b, c, fl = orc.velocity_update(v1[:, 0], v1[:, 1], v1[:, 2], np.arange(3, dtype=np.uint32), cs1, m1,
                                      np.tile(LANG(1.0), (3, 1)), 1.0, cfg, 0)
    assert np.array_equal(np.stack([a, b, c], 1), v1)
    assert fl.tolist() == [orc.FLAG_SKIPPED, orc.FLAG_SKIPPED, 0]


def test_ou_stationarity(orc):
    """Maxwellian cell + Langevin coefficients, mode 0, many steps: theta stays put in expectation and the velocity
    autocorrelation over one step is e^{-dt/tau}."""
    n, tau = 4000, 1.0
    rng = np.random.default_rng(6)
    v = rng.normal(0, math.sqrt(0.5), (n, 3)).astype(np.float32)
    cs = np.array([0, n], dtype=np.int32)
    pid = np.arange(n, dtype=np.uint32)
    cfg, _ = wl.couette()
    cfg.update(conserve_mode=0, dt=float(np.float32(0.25)), seed=1, eps2_scale=0.0)
    th, corr = [], []
    for step in range(40):
        mom = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 0)
        th.append((mom[0, 4] + mom[0, 7] + mom[0, 9]) / 3)
        vx, vy, vz, _ = orc.velocity_update(v[:, 0], v[:, 1], v[:, 2], pid, cs, mom, LANG(tau)[None, :], tau, cfg, step)
        new = np.stack([vx, vy, vz], 1)
        corr.append(np.corrcoef(v[:, 0] - v[:, 0].mean(), new[:, 0] - new[:, 0].mean())[0, 1])
        v = new
    assert abs(np.mean(th) - 0.5) < 0.02
    assert abs(np.mean(corr) - math.exp(-0.25)) < 0.01


# ------------------------------------------------------------------------------------------------ S7
def test_streaming_is_fp32_fma_and_walls_keep_particles_inside(orc):
    cfg, st = wl.cavity(20, 50, seed=2)
    cfg["dt"] = float(np.float32(0.05))                                  # large step: many wall hits
    out = orc.stream_walls(st, cfg, step=3)
    xmax = np.float32(cfg["x0"]) + np.float32(cfg["nx"]) * np.float32(cfg["dx"])
    assert out["x"].min() >= cfg["x0"] and out["x"].max() < xmax
    assert out["y"].min() >= cfg["y0"] and out["y"].max() < xmax
    assert out["x"].shape[0] == st["x"].shape[0] and np.array_equal(out["pid"], st["pid"])
    # particles that hit nothing: position is the single-rounding fused multiply-add, velocity untouched
    xe = (st["x"].astype(np.float64) + st["vx"].astype(np.float64) * np.float64(np.float32(cfg["dt"]))).astype(np.float32)
    ye = (st["y"].astype(np.float64) + st["vy"].astype(np.float64) * np.float64(np.float32(cfg["dt"]))).astype(np.float32)
    free = (xe >= cfg["x0"]) & (xe < xmax) & (ye >= cfg["y0"]) & (ye < xmax)
    assert 0.3 < free.mean() < 0.99
    assert np.array_equal(out["x"][free], xe[free]) and np.array_equal(out["y"][free], ye[free])
    for k in ("vx", "vy", "vz"):
        assert np.array_equal(out[k][free], st[k][free])
    # mirrored position of a left-wall hit: x <- xw + (xw - x)
    left = (xe < cfg["x0"]) & (ye >= cfg["y0"]) & (ye < xmax)
    assert left.sum() > 100
    np.testing.assert_array_equal(out["x"][left], np.float32(cfg["x0"]) + (np.float32(cfg["x0"]) - xe[left]))


def test_diffuse_wall_half_range_maxwellian(orc):
    """Re-emitted velocities: <v_n> = sqrt(pi theta_w / 2), <v_n^2> = 2 theta_w, tangential mean U_w, variance theta_w."""
    n, th_w, lid = 200_000, 0.8, 0.148
    walls = [(1, th_w, 0, 0, 0)] * 3 + [(1, th_w, lid, 0, -0.05)]
    cfg = wl.make_config(4, 4, 0.25, 0.25, 1.0, 1.0, walls, seed=11)
    rng = np.random.default_rng(0)
    st = dict(x=rng.uniform(0.1, 0.9, n).astype(np.float32), y=np.full(n, 0.9, np.float32),
              vx=np.zeros(n, np.float32), vy=np.full(n, 0.5, np.float32), vz=np.zeros(n, np.float32),
              pid=np.arange(n, dtype=np.uint32))
    out = orc.stream_walls(st, cfg, step=0)                              # every particle crosses the lid (y = 1)
    vn = -out["vy"].astype(np.float64)
    se = 5 / math.sqrt(n)
    assert np.all(vn > 0)
    assert abs(vn.mean() - math.sqrt(math.pi * th_w / 2)) < se * math.sqrt(th_w)
    assert abs((vn ** 2).mean() - 2 * th_w) < se * 2 * th_w
    assert abs(out["vx"].mean() - lid) < se * math.sqrt(th_w) and abs(out["vz"].mean() + 0.05) < se * math.sqrt(th_w)
    assert abs(out["vx"].var() - th_w) < se * 2 * th_w and abs(out["vz"].var() - th_w) < se * 2 * th_w
    np.testing.assert_array_equal(out["y"], np.float32(1.0) + (np.float32(1.0) - np.float32(1.4)))


def test_periodic_and_body(orc):
    walls = [(2, 0.5, 0, 0, 0)] * 2 + [(0, 0.5, 0, 0, 0)] * 2
    cfg = wl.make_config(8, 8, 1.0, 1.0, 1.0, 1.0, walls, seed=2, body=(4.0, 4.0, 2.0, 1.25))
    st = dict(x=np.float32([7.5, 0.5, 1.0, 3.0]), y=np.float32([1, 1, 4.0, 4.5]), vx=np.float32([1, -1, 1.5, 0]),
              vy=np.float32([0, 0, 0, 0]), vz=np.zeros(4, np.float32), pid=np.arange(4, dtype=np.uint32))
    out = orc.stream_walls(st, cfg, step=0)
    assert out["x"][0] == np.float32(0.5) and out["x"][1] == np.float32(7.5)     # wrapped
    r = np.hypot(out["x"][2:] - 4.0, out["y"][2:] - 4.0)
    assert np.all(r >= 2.0) and np.all(r < 2.0 * 1.00001)                         # pushed out to the surface
    vr = (out["vx"][2:] * (out["x"][2:] - 4) + out["vy"][2:] * (out["y"][2:] - 4)) / r
    assert np.all(vr > 0)                                                          # re-emitted outwards
