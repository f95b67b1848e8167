"""Pins for the oracle's exact cubic-FP closure (S2/S3).  CPU only.

None of these re-types the oracle's matrix: they check the SOLUTION against (1) the Langevin special case (PAPER.md
Eq. 4 :77, :174), (2) a linearised Grad-13 closed form consistent with Pr = 2/3 (:37, :87), (3) the relaxation
constraints of Eq. 3 (:69) evaluated directly from particles with the drift of Eq. 8 (:102), (4) the conservation
identities <N_i> = 0 and <c.N> = 0 of Eq. 14/15 (:171-178), (5) residual / Cramer brute force / symmetries, and the
blocks V (rows 1-4) and W exactly as Table 1 prints them (:132, :136; tests/golden/table1_VW.txt).
"""
import os

import numpy as np
import pytest

from paper_2606_15622_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
S2 = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
S3 = [(0, 0, 0), (0, 0, 1), (0, 0, 2), (0, 1, 1), (0, 1, 2), (0, 2, 2), (1, 1, 1), (1, 1, 2), (1, 2, 2), (2, 2, 2)]


def record_from_tensors(N, U, P, t, F4, g):
    """FULL record from full tensors P[3,3], t[3,3,3], F4[3,3] (= <c^2 c_i c_j>), g[3]."""
    return np.array([N, *U] + [P[i, j] for i, j in S2] + [t[i, j, k] for i, j, k in S3] + [F4[i, j] for i, j in S2]
                    + list(g), dtype=np.float64)


def particle_tensors(c):
    n = c.shape[0]
    c2 = (c ** 2).sum(1)
    P = np.einsum("pi,pj->ij", c, c) / n
    t = np.einsum("pi,pj,pk->ijk", c, c, c) / n
    F4 = np.einsum("p,pi,pj->ij", c2, c, c) / n
    g = np.einsum("p,pi->i", c2 ** 2, c) / n
    return P, t, F4, g


def grad13_cell(n, seed, amp=1.0):
    cfg, st, ex = wl.grad13_cells(1, 1, n, seed=seed, smax=0.3 * amp, qmax=0.2 * amp)
    v = np.stack([st["vx"], st["vy"], st["vz"]], 1)
    return v


def test_langevin_special_case(orc):
    """Exact Maxwellian moments => c = -delta/tau, gamma = 0 exactly (eps^2 vanishes since P = theta I)."""
    for theta, tau in [(0.5, 1.0), (3.7, 0.13), (1e-3, 40.0)]:
        m = record_from_tensors(100, [1, 2, 3], theta * np.eye(3), np.zeros((3, 3, 3)), 5 * theta ** 2 * np.eye(3),
                                np.zeros(3))
        coef, flags, kappa = orc.closure_exact(m[None, :], tau)
        assert flags[0] == 0
        np.testing.assert_allclose(coef[0], [-1 / tau, 0, 0, -1 / tau, 0, -1 / tau, 0, 0, 0], rtol=0, atol=1e-14 / tau)
        assert 1 <= kappa[0] < 50


def _grad13_record(theta, s, q, tau):
    I = np.eye(3)
    P = theta * (I + s)
    t = np.zeros((3, 3, 3))
    for i in range(3):
        for j in range(3):
            for k in range(3):
                t[i, j, k] = 0.4 * (q[i] * I[j, k] + q[j] * I[i, k] + q[k] * I[i, j])
    F4 = 5 * theta ** 2 * I + 7 * theta ** 2 * s
    g = 28 * theta * q
    return record_from_tensors(50, [0, 0, 0], P, t, F4, g)


def test_linearised_grad13_closed_form(orc):
    """eps^2 = 0, moments of f_M[1 + pi_ij c_i c_j/(2 p theta) + 2/(5 p theta) q_i c_i (c^2/(2 theta) - 5/2)]:
    to first order c_ij = -delta_ij/tau and gamma_i = h_i/(6 tau theta^2) = q_i/(3 tau rho theta^2); the error is
    second order in the perturbation (checked: 10x smaller perturbation -> 100x smaller error)."""
    rng = np.random.default_rng(0)
    theta, tau = 0.7, 0.9
    a = rng.uniform(-1, 1, (3, 3))
    s0 = 0.5 * (a + a.T)
    s0 -= np.eye(3) * np.trace(s0) / 3
    q0 = rng.uniform(-1, 1, 3) * theta ** 1.5
    errs = []
    for amp in (1e-3, 1e-4):
        m = _grad13_record(theta, amp * s0, amp * q0, tau)
        coef, flags, _ = orc.closure_exact(m[None, :], tau, eps2_scale=0.0)
        assert flags[0] == 0
        expect = np.array([-1 / tau, 0, 0, -1 / tau, 0, -1 / tau, *(2 * amp * q0 / (6 * tau * theta ** 2))])
        # compare gamma relative to its own size, c relative to 1/tau
        e_c = np.max(np.abs(coef[0, :6] - expect[:6])) * tau
        e_g = np.max(np.abs(coef[0, 6:] - expect[6:])) / np.max(np.abs(expect[6:]))
        errs.append((e_c, e_g))
    assert errs[0][0] < 5e-3 and errs[0][1] < 5e-3       # c error is O(amp) (first-order stress coupling), gamma O(amp)
    assert errs[1][1] < errs[0][1] / 5                   # relative gamma error shrinks ~linearly => absolute quadratically


@pytest.mark.parametrize("eps2_scale", [0.0, 1.0, 5.0])
def test_substitution_into_relaxation_constraints(orc, eps2_scale):
    """Bypass the matrix: evaluate the drift A(c_p) of Eq. 8 for every particle with the solved coefficients and check
    d<c_i c_j>/dt = -(2/tau)(P_ij - theta delta_ij) and d<c_i c^2>/dt = -(4/(3 tau)) h_i  (Eq. 3 with Maxwell rates)."""
    tau = 0.37
    v = grad13_cell(400, seed=21) * 1.3 + [0.4, -0.1, 0.2]
    v = v.astype(np.float32)
    cs = np.array([0, v.shape[0]], dtype=np.int32)
    mom = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 1)
    coef, flags, kappa = orc.closure_exact(mom, tau, eps2_scale=eps2_scale)
    assert flags[0] == 0
    y = coef[0]
    Cm = np.array([[y[0], y[1], y[2]], [y[1], y[3], y[4]], [y[2], y[4], y[5]]])
    gam = y[6:]
    c = v.astype(np.float64) - v.astype(np.float64).mean(0)
    n = c.shape[0]
    c2 = (c ** 2).sum(1)
    P = c.T @ c / n
    theta = np.trace(P) / 3
    h = (c2[:, None] * c).mean(0)
    eps2 = eps2_scale * abs(np.linalg.det(P - theta * np.eye(3))) / (tau * theta ** 4)       # reading R2-e
    A = c @ Cm.T + gam[None, :] * (c2 - 3 * theta)[:, None] - eps2 * (c * c2[:, None] - h[None, :])
    lhs2 = (A.T @ c + c.T @ A) / n + 2 * theta / tau * np.eye(3)
    rhs2 = -(2 / tau) * (P - theta * np.eye(3))
    lhs3 = (A * c2[:, None]).mean(0) + 2 * ((A * c).sum(1)[:, None] * c).mean(0)
    rhs3 = -(4 / (3 * tau)) * h
    tol = 1e-15 * max(kappa[0], 10) * 50
    assert np.max(np.abs(lhs2 - rhs2)) < tol * theta / tau
    assert np.max(np.abs(lhs3 - rhs3)) < tol * theta ** 1.5 / tau
    # conservation identities of the exact closure (pin 4): <N_i> = 0 and <c.N> = 0, hence alpha^2 >= 1
    Nn = A + c / tau
    assert np.max(np.abs(Nn.mean(0))) < tol * np.sqrt(theta) / tau
    assert abs((Nn * c).sum(1).mean()) < tol * theta / tau


def test_residual_cramer_and_numpy_solve(orc):
    rng = np.random.default_rng(4)
    for seed in range(5):
        v = grad13_cell(60 + 40 * seed, seed=100 + seed).astype(np.float32)
        cs = np.array([0, v.shape[0]], dtype=np.int32)
        m = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 1)[0]
        tau = float(rng.uniform(0.1, 3))
        coef, flag, kappa, A, b = orc.closure_exact_system(m, tau)
        theta = (m[4] + m[7] + m[9]) / 3
        yhat = np.concatenate([coef[:6] * tau, coef[6:] * tau * np.sqrt(theta)])
        assert np.linalg.norm(A @ yhat - b) / np.linalg.norm(b) < 1e-12
        # Cramer's rule, brute force with numpy determinants
        d = np.linalg.det(A)
        cram = np.array([np.linalg.det(np.column_stack([A[:, :k], b, A[:, k + 1:]])) for k in range(9)]) / d
        np.testing.assert_allclose(yhat, cram, rtol=1e-9 * max(kappa, 1), atol=1e-12)
        np.testing.assert_allclose(yhat, np.linalg.solve(A, b), rtol=1e-10 * max(kappa, 1), atol=1e-13)
        assert kappa == pytest.approx(np.linalg.cond(A, 1), rel=1e-8)


def test_table1_blocks_as_printed(orc):
    """theta = tau = 1 so that the oracle's scaled matrix equals the unscaled one; compare V rows 1-4 and all of W
    with the entries printed in PAPER.md Table 1."""
    v = grad13_cell(500, seed=9).astype(np.float64)
    c = v - v.mean(0)
    c /= np.sqrt((c ** 2).sum(1).mean() / 3)           # theta = 1 exactly up to round-off
    P, t, F4, g = particle_tensors(c)
    m = record_from_tensors(500, [0, 0, 0], P, t, F4, g)
    _, flag, _, A, b = orc.closure_exact_system(m, 1.0, eps2_scale=0.0)
    h = np.einsum("ikk->i", t)
    env = {"P11": P[0, 0], "P12": P[0, 1], "P13": P[0, 2], "P22": P[1, 1], "P23": P[1, 2], "P33": P[2, 2],
           "h1": h[0], "h2": h[1], "h3": h[2]}
    checked = 0
    for line in open(os.path.join(GOLD, "table1_VW.txt")):
        if line.strip() and not line.startswith("#"):
            r, col, expr = line.split()
            assert A[int(r) - 1, int(col) - 1] == pytest.approx(eval(expr, {}, env), rel=1e-12, abs=1e-13), line
            checked += 1
    assert checked == 42
    # rows 5, 6 of V (garbled in the paper): the (2,3) and (3,3) instances of c_ik P_kj + c_jk P_ki (reading R2-c)
    np.testing.assert_allclose(A[4, :6], [0, P[0, 2], P[0, 1], P[1, 2], P[2, 2] + P[1, 1], P[1, 2]], atol=1e-13)
    np.testing.assert_allclose(A[5, :6], [0, 0, 2 * P[0, 2], 0, 2 * P[1, 2], 2 * P[2, 2]], atol=1e-13)


def test_axis_permutation_and_scaling(orc):
    v = (grad13_cell(300, seed=33) + [0.1, 0.2, 0.3]).astype(np.float32)
    cs = np.array([0, 300], dtype=np.int32)
    tau = 0.8

    def solve(vv, tt):
        m = orc.cell_moments(vv[:, 0].copy(), vv[:, 1].copy(), vv[:, 2].copy(), cs, 1)
        coef, flags, kap = orc.closure_exact(m, tt)
        assert flags[0] == 0
        y = coef[0]
        return np.array([[y[0], y[1], y[2]], [y[1], y[3], y[4]], [y[2], y[4], y[5]]]), y[6:], kap[0]
    C0, g0, kap = solve(v, tau)
    perm = [2, 0, 1]
    C1, g1, _ = solve(v[:, perm], tau)
    np.testing.assert_allclose(C1, C0[np.ix_(perm, perm)], rtol=1e-9 * kap, atol=1e-12)
    np.testing.assert_allclose(g1, g0[perm], rtol=1e-9 * kap, atol=1e-12)
    lam, mu = 4.0, 0.25                                  # powers of two: the scaled ensemble is exact in fp32
    C2, g2, _ = solve(v * np.float32(lam), tau * mu)
    np.testing.assert_allclose(C2, C0 / mu, rtol=1e-9 * kap)
    np.testing.assert_allclose(g2, g0 / (lam * mu), rtol=1e-9 * kap)


def test_flags_and_fallbacks(orc):
    theta, tau = 0.5, 2.0
    ok = record_from_tensors(100, [0, 0, 0], theta * np.eye(3), np.zeros((3, 3, 3)), 5 * theta ** 2 * np.eye(3),
                             np.zeros(3))
    empty = np.zeros(29)
    low = ok.copy(); low[0] = 9
    cold = ok.copy(); cold[4:] = 0                        # theta = 0
    sing = ok.copy(); sing[20:26] = [15 * theta ** 2 / 3 * 0.6, 0, 0, 15 * theta ** 2 / 3 * 0.6, 0, 15 * theta ** 2 / 3 * 0.6]
    # F = 9 theta^2 and F_ij = 3 theta P_ij  =>  Z = 0: the heat-flux block is singular
    coef, flags, kappa = orc.closure_exact(np.stack([ok, empty, low, cold, sing]), tau)
    lang = [-0.5, 0, 0, -0.5, 0, -0.5, 0, 0, 0]
    assert flags.tolist() == [0, orc.FLAG_EMPTY, orc.FLAG_LOWCOUNT, orc.FLAG_SINGULAR, orc.FLAG_SINGULAR]
    np.testing.assert_allclose(coef[0], lang, atol=1e-15)
    assert np.all(coef[1] == 0)
    for k in (2, 3, 4):
        assert coef[k].tolist() == lang


def test_c2_workload_condition_numbers(orc):
    """The C2 recipe (50 ppc) must produce solvable cells with a spread of condition numbers."""
    cfg, st, _ = wl.grad13_cells(12, 12, 50, seed=1)
    cs = (np.arange(145) * 50).astype(np.int32)
    mom = orc.cell_moments(st["vx"], st["vy"], st["vz"], cs, 1)
    coef, flags, kappa = orc.closure_exact(mom, 1.0)
    assert np.all(np.isfinite(coef))
    assert np.count_nonzero(flags & orc.FLAG_SINGULAR) == 0
    assert np.median(kappa) < 1e4
    # magnitude sanity: coefficients are O(1/tau) in nondimensional units for well-conditioned cells
    good = kappa < 1e3
    assert good.sum() > 50 and np.median(np.abs(coef[good, 0] + 1.0)) < 2.0
