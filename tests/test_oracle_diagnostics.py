"""Pins for the oracle's NEXT-2 sampling outputs (orc_cell_diagnostics, orc_average_results).  CPU only.

Each pin is something other than the oracle itself: hand values on octahedral point sets (derived in the comments),
numpy's slogdet for D_G (Eq. 22 :651), invariance under rotations of the velocity frame (catches a wrong
index, multiplicity or sign in the determinant and the tensor norms), the Maxwellian limits the paper names
(:415 Delta_4 -> 0; <c_i c_j c^2> -> 5 theta^2 delta_ij; D_G -> 0), D_G >= 0 (arithmetic-geometric mean), Eq. 20 by hand,
and the arithmetic mean for the running average (:217-219).
"""
import numpy as np
import pytest

NAMES = ["theta", "d4", "d4n", "DG", "Dq", "dseq", "dskin", "sig", "q", "m3", "R11", "R12", "R13", "R22", "R23", "R33"]


def _diag_of(orc, v, **kw):
    v = np.asarray(v, dtype=np.float32)
    cs = np.array([0, v.shape[0]], dtype=np.int32)
    m = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 1)
    return dict(zip(NAMES, orc.cell_diagnostics(m, **kw)[0])), m[0]


def _octa(a, b, c, shift=(0.0, 0.0, 0.0)):
    p = np.array([[a, 0, 0], [-a, 0, 0], [0, b, 0], [0, -b, 0], [0, 0, c], [0, 0, -c]], dtype=np.float64)
    return p + np.asarray(shift)


def test_hand_octahedron(orc):
    # six particles at +-a on the axes: P = a^2/3 I, theta = a^2/3, <c^4> = a^4, <c_i c_j c^2> = a^4/3 delta_ij, odd
    # moments vanish.  Delta_4 = a^4 - 15 a^4/9 = -2 a^4/3; /(15 theta^2) = -2/5; R_ii/(5 theta^2) = 3/5; D_G = 0.
    a = 2.0
    d, _ = _diag_of(orc, _octa(a, a, a, shift=(4.0, -1.0, 0.5)), theta_inf=a * a / 6.0, n_inf=2.0)
    assert d["theta"] == pytest.approx(a * a / 3, rel=1e-12)
    assert d["d4"] == pytest.approx(-2 * a ** 4 / 3, rel=1e-12)
    assert d["d4n"] == pytest.approx(-0.4, rel=1e-12)
    assert d["DG"] == pytest.approx(0.0, abs=1e-12) and d["Dq"] == pytest.approx(0.0, abs=1e-12)
    assert d["sig"] == pytest.approx(0.0, abs=1e-12) and d["m3"] == pytest.approx(0.0, abs=1e-12)
    for k in ("R11", "R22", "R33"):
        assert d[k] == pytest.approx(0.6, rel=1e-12)
    for k in ("R12", "R13", "R23"):
        assert d[k] == pytest.approx(0.0, abs=1e-12)
    # Eq. 20 by hand: theta = 2 theta_inf, N = 3 n_inf
    assert d["dseq"] == pytest.approx(1.5 * np.log(2.0) - np.log(3.0), rel=1e-12)
    assert d["dskin"] == pytest.approx(d["dseq"], rel=1e-12)


def test_hand_anisotropic(orc):
    # +-a, +-b, +-c on the axes: P = diag(a^2, b^2, c^2)/3, theta = (a^2+b^2+c^2)/9,
    # D_G = -1/2 log(a^2 b^2 c^2 / (27 theta^3)); sigma_norm = sqrt(sum (P_ii - theta)^2)/theta; <c^4> = (a^4+b^4+c^4)/3
    a, b, c = 1.0, 2.0, 3.0
    d, _ = _diag_of(orc, _octa(a, b, c), dg_inf=0.25)
    th = (a * a + b * b + c * c) / 9
    assert d["theta"] == pytest.approx(th, rel=1e-12)
    dg = -0.5 * np.log(a * a * b * b * c * c / 27 / th ** 3)
    assert d["DG"] == pytest.approx(dg, rel=1e-12) and dg > 0
    assert d["dskin"] == pytest.approx(d["dseq"] - (dg - 0.25), rel=1e-12)
    sig = np.sqrt(sum((x * x / 3 - th) ** 2 for x in (a, b, c))) / th
    assert d["sig"] == pytest.approx(sig, rel=1e-12)
    assert d["d4"] == pytest.approx((a ** 4 + b ** 4 + c ** 4) / 3 - 15 * th * th, rel=1e-12)
    assert d["R22"] == pytest.approx(b ** 4 / 3 / (5 * th * th), rel=1e-12)


def test_hand_third_order(orc):
    # two particles at (2a,0,0), four at (-a,0,0): mean 0, c_x only; <c^2> = (2*4+4)/6 a^2 = 2 a^2, <c^3> = (2*8-4)/6 a^3
    # = 2 a^3: theta = 2a^2/3, h = (2a^3,0,0), q_hat = 2a^3/(2 theta^1.5), t_111 = 2a^3 -> m3_norm = 2a^3/theta^1.5.
    # The covariance is singular: D_G = +inf and ds_kin,G = -inf.
    a = 0.7
    v = [[2 * a, 0, 0]] * 2 + [[-a, 0, 0]] * 4
    d, _ = _diag_of(orc, v)
    th = 2 * a * a / 3
    assert d["theta"] == pytest.approx(th, rel=1e-6)
    assert d["q"] == pytest.approx(2 * a ** 3 / (2 * th ** 1.5), rel=1e-6)
    assert d["Dq"] == pytest.approx(d["q"] ** 2 / 5, rel=1e-12)
    assert d["m3"] == pytest.approx(2 * a ** 3 / th ** 1.5, rel=1e-6)
    assert d["DG"] == np.inf and d["dskin"] == -np.inf


def test_dg_matches_slogdet_and_is_nonnegative(orc):
    rng = np.random.default_rng(5)
    for n in (5, 17, 400):
        A = rng.normal(size=(3, 3))
        v = rng.normal(size=(n, 3)) @ A.T + rng.normal(size=3)
        d, m = _diag_of(orc, v)
        P = np.array([[m[4], m[5], m[6]], [m[5], m[7], m[8]], [m[6], m[8], m[9]]])
        sign, logdet = np.linalg.slogdet(P / d["theta"])
        assert sign > 0
        assert d["DG"] == pytest.approx(-0.5 * logdet, rel=1e-10, abs=1e-12)
        assert d["DG"] >= -1e-14


def test_rotation_invariance(orc):
    rng = np.random.default_rng(11)
    v = rng.normal(size=(60, 3)) * np.array([0.5, 1.0, 1.7]) + rng.gamma(2.0, size=(60, 3)) * 0.3
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    d0, _ = _diag_of(orc, v)
    d1, _ = _diag_of(orc, v @ Q.T)
    for k in ("theta", "d4", "d4n", "DG", "Dq", "sig", "q", "m3"):
        assert d1[k] == pytest.approx(d0[k], rel=2e-5), k          # fp32 inputs are re-rounded after the rotation
    # the trace of R_norm is invariant: sum R_ii = <c^4> / (5 theta^2)
    assert d1["R11"] + d1["R22"] + d1["R33"] == pytest.approx(d0["R11"] + d0["R22"] + d0["R33"], rel=2e-5)
    R0 = np.array([[d0["R11"], d0["R12"], d0["R13"]], [d0["R12"], d0["R22"], d0["R23"]], [d0["R13"], d0["R23"], d0["R33"]]])
    R1 = np.array([[d1["R11"], d1["R12"], d1["R13"]], [d1["R12"], d1["R22"], d1["R23"]], [d1["R13"], d1["R23"], d1["R33"]]])
    assert np.allclose(Q @ R0 @ Q.T, R1, rtol=0, atol=5e-5)


def test_maxwellian_limits(orc):
    # Delta_4 is the excess over a local Maxwellian; n = 4e5 samples: statistical error ~ few / sqrt(n)
    rng = np.random.default_rng(2)
    n = 400000
    v = rng.normal(scale=np.sqrt(0.5), size=(n, 3)) + np.array([0.3, -0.2, 9.0])
    d, _ = _diag_of(orc, v)
    assert d["theta"] == pytest.approx(0.5, rel=5e-3)
    assert abs(d["d4n"]) < 0.02 and d["DG"] < 1e-4 and d["Dq"] < 1e-4 and d["sig"] < 0.01 and d["m3"] < 0.02
    for k in ("R11", "R22", "R33"):
        assert d[k] == pytest.approx(1.0, abs=0.02)
    for k in ("R12", "R13", "R23"):
        assert abs(d[k]) < 0.01


def test_empty_and_cold_cells(orc):
    m = np.zeros((2, 29))
    m[1, 0] = 3.0                       # three particles at rest: theta = 0
    assert (orc.cell_diagnostics(m) == 0).all()


def test_running_average_is_the_mean(orc):
    rng = np.random.default_rng(9)
    xs = rng.normal(size=(7, 5, 16))
    avg = np.zeros((5, 16))
    for k in range(7):
        orc.average_results(xs[k], k, avg)
        assert np.allclose(avg, xs[: k + 1].mean(axis=0), rtol=1e-13, atol=1e-15)


def test_dm6_hand_and_maxwellian(orc):
    # octahedron: every particle has c^2 = a^2 -> DM6 = a^6 exactly (any bulk velocity);  2 + 4 points on a line:
    # c = 2a (x2), -a (x4): <c^6> = (2 * 64 + 4) / 6 a^6 = 22 a^6;  Maxwellian: <c^6> = 105 theta^3 (chi-square with 3
    # degrees of freedom: E[r^6] = 3 * 5 * 7 theta^3)
    a = 1.5
    v = _octa(a, a, a, shift=(3.0, 0.25, -7.0)).astype(np.float32)
    cs = np.array([0, 6], dtype=np.int32)
    assert orc.cell_dm6(v[:, 0], v[:, 1], v[:, 2], cs)[0] == pytest.approx(a ** 6, rel=1e-6)
    b = 0.5
    w = np.array([[2 * b, 0, 0]] * 2 + [[-b, 0, 0]] * 4, dtype=np.float32)
    assert orc.cell_dm6(w[:, 0], w[:, 1], w[:, 2], cs)[0] == pytest.approx(22 * b ** 6, rel=1e-6)
    rng = np.random.default_rng(3)
    n = 400000
    g = (rng.normal(scale=np.sqrt(0.5), size=(n, 3)) + np.array([1.0, 2.0, -3.0])).astype(np.float32)
    got = orc.cell_dm6(g[:, 0], g[:, 1], g[:, 2], np.array([0, 0, n], dtype=np.int32))
    assert got[0] == 0.0                                            # empty cell
    assert got[1] == pytest.approx(105 * 0.5 ** 3, rel=0.03)        # relative sd of the estimate ~ 10 / sqrt(n)


def test_three_particle_cell_is_defined_singular(orc):
    """Reading R10: a cell with N < 4 has a covariance of rank <= N - 1, so D_G = +inf and ds_kin,G = -inf whatever the
    rounding of its (mathematically zero) determinant says; N = 4 in general position is regular.  theta > 0 in both."""
    # three-particle sets whose rank-2 covariance has a determinant that ROUNDS to a small positive number in fp64
    # (found by search): without the N < 4 rule they would report a finite D_G ~ 19
    for v3 in ([[0.1, -0.1, 0.4], [0.1, -0.3, 0.2], [0.8, 0.6, -0.4]],
               [[-0.6, -0.3, 0.1], [-0.6, -0.1, -0.1], [0.3, 0.1, 0.2]],
               [[0.3, -0.2, 0.5], [-0.4, 0.6, 0.1], [0.2, 0.1, -0.7]]):
        d3, m3 = _diag_of(orc, np.float32(v3))
        assert m3[0] == 3 and d3["theta"] > 0.05
        assert d3["DG"] == np.inf and d3["dskin"] == -np.inf
        assert np.isfinite(d3["d4"]) and np.isfinite(d3["sig"]) and np.isfinite(d3["dseq"])
    v4 = np.float32([[0.3, -0.2, 0.5], [-0.4, 0.6, 0.1], [0.2, 0.1, -0.7], [-0.1, -0.5, 0.1]])
    d4, m4 = _diag_of(orc, v4)
    c = v4.astype(np.float64) - v4.astype(np.float64).mean(0)
    Th = c.T @ c / 4
    sign, logdet = np.linalg.slogdet(Th / (np.trace(Th) / 3))
    assert sign > 0 and d4["DG"] == pytest.approx(-0.5 * logdet, rel=1e-10)
