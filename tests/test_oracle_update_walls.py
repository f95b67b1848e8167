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


# ------------------------------------------------------------------------------------------------ Eq. 14 pins
def _recover_N(orc, v, cs, pid, mom, coef, tau, cfg, step, alpha):
    """N_i per particle from the oracle's OUTPUT of a conserve_mode-0 update, by inverting Eq. 13:
    N = (alpha c* - c E1 - sqrt(theta (1 - E2)) xi) / ((1 - E1) tau), with the separately pinned normals."""
    vx, vy, vz, fl = orc.velocity_update(v[:, 0], v[:, 1], v[:, 2], pid, cs, mom, coef[None, :], np.float32(tau), cfg, step)
    assert fl[0] == 0
    U, theta = mom[0, 1:4], (mom[0, 4] + mom[0, 7] + mom[0, 9]) / 3
    tau32 = float(np.float32(tau))
    a = cfg["dt"] / tau32
    E1, E2 = math.exp(-a), math.exp(-2 * a)
    xi = orc.normals(pid, step, 0, cfg["seed"])
    cstar = np.stack([vx, vy, vz], 1).astype(np.float64) - U
    c = v.astype(np.float64) - U
    w = c * E1 + math.sqrt(theta * (1 - E2)) * xi
    kap = (1 - E1) * tau32
    if alpha is None:
        return cstar, w, kap, c, theta, (E1, E2, tau32)
    return (alpha * cstar - w) / kap, c, theta, (E1, E2, tau32)


def _eq14_numpy(c, theta, P, h, coef, tau, eps2_scale):
    """Eq. 14 typed out: N_i = (C_ij + delta_ij/tau) c_j + gam_i (c^2 - 3 theta) - eps2 (c_i c^2 - h_i),
    C symmetric from (c11, c12, c13, c22, c23, c33), eps2 = eps2_scale |det(P - theta I)| / (tau theta^4) (R2-e)."""
    C = np.array([[coef[0], coef[1], coef[2]], [coef[1], coef[3], coef[4]], [coef[2], coef[4], coef[5]]], dtype=np.float64)
    gam = np.asarray(coef[6:9], dtype=np.float64)
    Pm = np.array([[P[0], P[1], P[2]], [P[1], P[3], P[4]], [P[2], P[4], P[5]]])
    eps2 = eps2_scale * abs(np.linalg.det(Pm - theta * np.eye(3))) / (tau * theta ** 4)
    c2 = (c ** 2).sum(1)
    return c @ (C + np.eye(3) / tau).T + gam[None, :] * (c2 - 3 * theta)[:, None] - eps2 * (c * c2[:, None] - h[None, :])


@pytest.mark.parametrize("eps2_scale", [1.0, 5.0])
def test_update_drift_matches_eq14(orc, eps2_scale):
    """The non-Langevin drift inside the update, per particle, against Eq. 14 written out in numpy: nine distinct
    coefficients (no accidental symmetry), theta != 1 (so a lost 1/theta^4 shows), eps2 > 0."""
    cfg, v, cs, pid = _cell(orc, 400, 21)
    v = (v * np.float32(1.3)).astype(np.float32)                          # theta ~ 0.85
    cfg.update(conserve_mode=0, eps2_scale=float(np.float32(eps2_scale)), dt=float(np.float32(0.2)), seed=13)
    tau = 0.8
    mom = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 1)
    coef = np.float32([-1.1, 0.23, -0.31, -0.87, 0.12, -1.4, 0.07, -0.05, 0.11]) / np.float32(tau)
    U, P = mom[0, 1:4], mom[0, 4:10]
    theta = (P[0] + P[3] + P[5]) / 3
    t = mom[0, 10:20]                                                     # 111,112,113,122,123,133,222,223,233,333
    h = np.array([t[0] + t[3] + t[5], t[1] + t[6] + t[8], t[2] + t[7] + t[9]])
    c = v.astype(np.float64) - U
    tau32 = float(np.float32(tau))
    N_ref = _eq14_numpy(c, theta, P, h, coef.astype(np.float64), tau32, cfg["eps2_scale"])
    assert np.abs(N_ref - c @ (np.diag([1 / tau32] * 3) + np.diag(coef[[0, 3, 5]].astype(np.float64))).T).max() > 0.05
    a = cfg["dt"] / tau32
    E1, E2 = math.exp(-a), math.exp(-2 * a)
    alpha2 = 1 + tau32 / (3 * theta) * (tau32 * (1 - E1) ** 2 * (N_ref ** 2).sum(1).mean()
                                        + 2 * (E1 - E2) * (c * N_ref).sum(1).mean())          # Eq. 15 (:178)
    N_got, _, _, _ = _recover_N(orc, v, cs, pid, mom, coef, tau, cfg, 7, math.sqrt(alpha2))
    # output velocities are fp32: |dN| <~ 6e-8 |v| alpha / ((1 - E1) tau)
    np.testing.assert_allclose(N_got, N_ref, atol=3e-7 * np.abs(v).max() / ((1 - E1) * tau32))
    assert abs(N_got.mean(0)).max() < 1e-6                                # <N_i> = 0 for any coefficients


def test_update_drift_satisfies_closure_constraints(orc):
    """Independent of any retyped Eq. 14: with the EXACT closure's coefficients the drift the update applies must
    reproduce the relaxation rates the closure imposes (Eq. 3 :69, :124; oracle header):
      <N_i c_j + N_j c_i> = <A_i c_j + A_j c_i> + 2 P_ij / tau = 0                     (stress rate 2/tau)
      <N_i c^2 + 2 c_i c.N> = -(4/(3 tau)) h_i + 3 h_i / tau = (5/(3 tau)) h_i         (heat-flux rate 4/(3 tau))
    where A = N - c/tau is the drift of Eq. 8 and the diffusion terms (2 theta/tau delta_ij; <c_i> = 0) are moved to
    the right.  alpha is not assumed: it is fixed by the trace of the first identity, <c.N> = 0, and must then satisfy
    Eq. 15 with the recovered N."""
    cfg, st, _ = wl.grad13_cells(1, 1, 3000, seed=31, smax=0.25, qmax=0.15)
    v = (np.stack([st["vx"], st["vy"], st["vz"]], 1) * np.float32(1.2) + np.float32([0.4, -0.1, 0.2])).astype(np.float32)
    cs = np.array([0, v.shape[0]], dtype=np.int32)
    pid = st["pid"]
    tau = 0.9
    cfg.update(conserve_mode=0, eps2_scale=float(np.float32(2.0)), dt=float(np.float32(0.25)), seed=4)
    mom = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 1)
    coef, flags, kappa = orc.closure_exact(mom, float(np.float32(tau)), cfg["eps2_scale"])
    assert flags[0] == 0 and kappa[0] < 1e4
    coef32 = coef[0].astype(np.float32)
    cstar, w, kap, c, theta, (E1, E2, tau32) = _recover_N(orc, v, cs, pid, mom, coef32, tau, cfg, 3, None)
    alpha = (c * w).sum(1).mean() / (c * cstar).sum(1).mean()             # from <c.N> = 0
    N = (alpha * cstar - w) / kap
    alpha2_eq15 = 1 + tau32 / (3 * theta) * (tau32 * (1 - E1) ** 2 * (N ** 2).sum(1).mean() + 2 * (E1 - E2) * (c * N).sum(1).mean())
    assert abs(alpha * alpha - alpha2_eq15) < 1e-5                         # fp32 coefficients and velocities
    assert alpha > 1.0                                                     # Eq. 15 with <c.N> = 0: alpha^2 = 1 + (...) <N.N>
    S = np.einsum("pi,pj->ij", N, c) / c.shape[0]
    S = S + S.T
    scale = theta / tau32
    assert np.abs(S).max() < 2e-5 * scale, S / scale                       # all six stress identities
    t = mom[0, 10:20]
    h = np.array([t[0] + t[3] + t[5], t[1] + t[6] + t[8], t[2] + t[7] + t[9]])
    c2 = (c ** 2).sum(1)
    H = (N * c2[:, None] + 2 * c * (c * N).sum(1)[:, None]).mean(0)
    np.testing.assert_allclose(H, 5.0 / (3.0 * tau32) * h, atol=2e-4 * theta ** 1.5 / tau32)
    assert np.abs(h).max() > 0.01 * theta ** 1.5                           # the heat flux is not trivially zero


def test_two_particle_cell_is_updated(orc):
    """R5: a cell with N = 2 and theta > 0 is updated (only N < 2 or theta <= 0 is skipped): conserve_mode 1 keeps its
    momentum and energy and the velocities change."""
    v = np.float32([[0.3, -0.2, 0.5], [-0.4, 0.6, 0.1], [9, 9, 9]])
    cs = np.array([0, 2, 3], dtype=np.int32)
    cfg, _ = wl.couette()
    cfg.update(conserve_mode=1, seed=2, dt=float(np.float32(0.3)))
    mom = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 0)
    vx, vy, vz, fl = orc.velocity_update(v[:, 0], v[:, 1], v[:, 2], np.arange(3, dtype=np.uint32), cs, mom,
                                         np.tile(LANG(1.0), (2, 1)), 1.0, cfg, 0)
    new = np.stack([vx, vy, vz], 1).astype(np.float64)
    assert fl.tolist() == [0, orc.FLAG_SKIPPED]
    assert np.array_equal(new[2], v[2]) and np.abs(new[:2] - v[:2]).max() > 0.01
    old = v[:2].astype(np.float64)
    np.testing.assert_allclose(new[:2].mean(0), old.mean(0), atol=2e-7)
    np.testing.assert_allclose(((new[:2] - new[:2].mean(0)) ** 2).sum(), ((old - old.mean(0)) ** 2).sum(), rtol=1e-6)


# ------------------------------------------------------------------------------------------------ S7: x-walls
@pytest.mark.parametrize("side", [0, 1])
def test_couette_plate_reemission(orc, side):
    """BASELINE config 1 geometry: diffuse plates at xmin/xmax moving in y (and, to tell the
    tangential components apart, a different speed in z).  Every particle crosses the plate: v_x must point into the
    gas with the half-range law, <v_y> = U_w,y, <v_z> = U_w,z, tangential variances theta_w."""
    n, th_w = 200_000, 0.6
    uwy, uwz = (-0.3, 0.11) if side == 0 else (0.3, -0.17)
    walls = [(1, th_w, 0, -0.3, 0.11), (1, th_w, 0, 0.3, -0.17), (0, 0.5, 0, 0, 0), (0, 0.5, 0, 0, 0)]
    cfg = wl.make_config(8, 1, 0.125, 1.0, 1.0, 1.0, walls, seed=17)
    rng = np.random.default_rng(1)
    x0 = 0.1 if side == 0 else 0.9
    st = dict(x=np.full(n, x0, np.float32), y=rng.uniform(0.1, 0.9, n).astype(np.float32),
              vx=np.full(n, -0.5 if side == 0 else 0.5, np.float32), vy=np.full(n, 7.0, np.float32) * 0,
              vz=np.full(n, 3.0, np.float32), pid=np.arange(n, dtype=np.uint32))
    out = orc.stream_walls(st, cfg, step=2)
    vn = out["vx"].astype(np.float64) * (1.0 if side == 0 else -1.0)       # into the gas
    se = 5 / math.sqrt(n)
    assert np.all(vn > 0)
    assert abs(vn.mean() - math.sqrt(math.pi * th_w / 2)) < se * math.sqrt(th_w)
    assert abs((vn ** 2).mean() - 2 * th_w) < se * 2 * th_w
    assert abs(out["vy"].mean() - uwy) < se * math.sqrt(th_w) and abs(out["vz"].mean() - uwz) < se * math.sqrt(th_w)
    assert abs(out["vy"].var() - th_w) < se * 2 * th_w and abs(out["vz"].var() - th_w) < se * 2 * th_w
    xw = np.float32(0.0 if side == 0 else 1.0)
    xe = np.float32(x0) + np.float32(-0.5 if side == 0 else 0.5)            # exact in fp32
    np.testing.assert_array_equal(out["x"], xw + (xw - xe))
    assert np.array_equal(out["y"], st["y"])                                # vy = 0: y untouched, ny = 1


# ------------------------------------------------------------------------------------------------ S7: freestream reservoir
def _flux_maxwellian_moments(U, theta):
    """E[v], E[v^2] and the CDF of f(v) ~ v exp(-(v - U)^2 / (2 theta)) on v > 0 by plain quadrature (no sampler involved)."""
    sg = math.sqrt(theta)
    v = np.linspace(0.0, max(U, 0.0) + 12.0 * sg, 400001)
    f = v * np.exp(-(v - U) ** 2 / (2.0 * theta))
    dv = v[1] - v[0]
    Z = f.sum() * dv
    cdf = np.cumsum(f) * dv / Z
    return (f * v).sum() * dv / Z, (f * v * v).sum() * dv / Z, v, cdf


@pytest.mark.parametrize("U", [0.25, 9.09])
def test_reservoir_reinsertion(orc, U):
    """Reading R11: a particle leaving through a freestream face re-enters at xmin with the flux-
    weighted drifting half-Maxwellian in v_x (moments and CDF against quadrature), Gaussian tangentials about U_inf, a
    position uniform along the face and within one freestream step of it; the particle count is constant and every particle
    ends inside the domain.  Subsonic (many rejections) and Mach 10 (almost none)."""
    n, th = 200_000, 0.5
    walls = [(wl.WALL_INFLOW, th, U, -0.2, 0.1)] * 4
    cfg = wl.make_config(10, 8, 1.0, 0.5, 0.1, 1.0, walls, seed=23)
    rng = np.random.default_rng(3)
    # a quarter of the particles leaves through each face
    q = n // 4
    x = np.concatenate([np.full(q, 0.01), np.full(q, 9.99), rng.uniform(1, 9, q), rng.uniform(1, 9, q)]).astype(np.float32)
    y = np.concatenate([rng.uniform(0.5, 3.5, q), rng.uniform(0.5, 3.5, q), np.full(q, 0.01), np.full(q, 3.99)]).astype(np.float32)
    vx = np.concatenate([np.full(q, -1.0), np.full(q, 1.0), np.zeros(q), np.zeros(q)]).astype(np.float32)
    vy = np.concatenate([np.zeros(q), np.zeros(q), np.full(q, -1.0), np.full(q, 1.0)]).astype(np.float32)
    st = dict(x=x, y=y, vx=vx, vy=vy, vz=np.full(n, 7.0, np.float32), pid=np.arange(n, dtype=np.uint32))
    out = orc.stream_walls(st, cfg, step=4)
    assert out["x"].shape[0] == n and np.array_equal(out["pid"], st["pid"])
    pen = float(np.float32(np.float32(U) * np.float32(cfg["dt"])))
    assert out["x"].min() >= 0.0 and out["x"].max() <= pen * (1 + 1e-6) + 1e-7          # within one freestream step of xmin
    assert out["y"].min() >= 0.0 and out["y"].max() < 4.0
    se = 5 / math.sqrt(n)
    m1, m2, vg, cdf = _flux_maxwellian_moments(U, th)
    v = out["vx"].astype(np.float64)
    assert np.all(v > 0)
    assert abs(v.mean() - m1) < se * math.sqrt(m2 - m1 * m1) and abs((v * v).mean() - m2) < se * 3 * m2
    for qq in (0.01, 0.1, 0.5, 0.9, 0.99):                                              # CDF at five quantiles
        vq = vg[np.searchsorted(cdf, qq)]
        assert abs((v <= vq).mean() - qq) < se
    assert abs(out["vy"].mean() + 0.2) < se * math.sqrt(th) and abs(out["vz"].mean() - 0.1) < se * math.sqrt(th)
    assert abs(out["vy"].var() - th) < se * 2 * th and abs(out["vz"].var() - th) < se * 2 * th
    # positions: uniform along the face, uniform in the entry strip, independent of the face the particle left through
    assert abs(out["y"].mean() - 2.0) < se * 4 / math.sqrt(12) and abs(out["x"].mean() - pen / 2) < se * pen / math.sqrt(12) + 1e-7
    assert abs(np.corrcoef(out["y"], v)[0, 1]) < se and abs(np.corrcoef(out["x"], v)[0, 1]) < se
    # a particle that stays inside is not touched
    st2 = dict(st, x=np.full(n, 5.0, np.float32), y=np.full(n, 2.0, np.float32))
    out2 = orc.stream_walls(st2, cfg, step=4)
    assert np.array_equal(out2["vz"], st["vz"]) and np.array_equal(out2["vx"], st["vx"])
