"""Pins for the oracle's MLP surrogate (S4) and counter-based normals (S6).  CPU only."""
import math
import os

import numpy as np
import pytest

from paper_2606_15622_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------------------------------------ S4
def test_parameter_counts():
    """16-256-256-256-256-9 with biases has 204,041 parameters; BASELINE's 13-64-64-64-9 has 9,801."""
    for dims, count in [((16, 256, 256, 256, 256, 9), 204041), ((13, 64, 64, 64, 9), 9801)]:
        mlp = wl.xavier_mlp(dims, feature_set=1 if dims[0] == 16 else 0)
        assert sum(w.size for w in mlp["W"]) + sum(b.size for b in mlp["b"]) == count


def _mlp(dims, act=0):
    m = wl.xavier_mlp(dims, seed=3, act=act, bias_scale=0.5)
    return m


def test_hand_cases(orc):
    mlp = _mlp((13, 64, 64, 64, 9))
    x = np.linspace(-1, 1, 13).astype(np.float32)
    # all-zero weights: y = b_L * y_scale + y_mean
    z = dict(mlp)
    z["W"] = [np.zeros_like(w) for w in mlp["W"]]
    z["b"] = [np.zeros_like(b) for b in mlp["b"][:-1]] + [mlp["b"][-1]]
    y = orc.mlp_forward(z, x)
    np.testing.assert_allclose(y, mlp["b"][-1].astype(np.float64) * mlp["y_scale"] + mlp["y_mean"], rtol=1e-15)
    # one hidden unit, SiLU and ReLU, by hand
    for act in (0, 1):
        one = dict(dims=np.array([2, 1, 1], dtype=np.int32), W=[np.float32([[0.5, -2.0]]), np.float32([[3.0]])],
                   b=[np.float32([0.25]), np.float32([-1.0])], x_mean=np.float32([1, 2]), x_scale=np.float32([2, 4]),
                   y_mean=np.float32([10]), y_scale=np.float32([0.5]), act=act)
        xx = np.float32([3.0, -2.0])
        pre = 0.5 * (3 - 1) / 2 + (-2.0) * (-2 - 2) / 4 + 0.25          # = 2.75
        hid = pre / (1 + math.exp(-pre)) if act == 0 else max(pre, 0.0)
        assert orc.mlp_forward(one, xx)[0] == pytest.approx((3.0 * hid - 1.0) * 0.5 + 10, rel=1e-15)
        xx = np.float32([-3.0, 6.0])                                     # pre = -1 - 2 + 0.25 = -2.75
        pre = 0.5 * (-3 - 1) / 2 + (-2.0) * (6 - 2) / 4 + 0.25
        hid = pre / (1 + math.exp(-pre)) if act == 0 else 0.0
        assert orc.mlp_forward(one, xx)[0] == pytest.approx((3.0 * hid - 1.0) * 0.5 + 10, rel=1e-15)
    # identity-like ReLU net on positive inputs passes the input through
    eye = dict(dims=np.array([9, 9, 9], dtype=np.int32), W=[np.eye(9, dtype=np.float32)] * 2,
               b=[np.zeros(9, np.float32)] * 2, x_mean=np.zeros(9, np.float32), x_scale=np.ones(9, np.float32),
               y_mean=np.zeros(9, np.float32), y_scale=np.ones(9, np.float32), act=1)
    xx = np.arange(1, 10, dtype=np.float32)
    np.testing.assert_array_equal(orc.mlp_forward(eye, xx), xx.astype(np.float64))


def test_independent_numpy_forward_and_head_linearity(orc):
    rng = np.random.default_rng(0)
    for dims, act in [((13, 64, 64, 64, 9), 0), ((16, 256, 256, 256, 256, 9), 1), ((13, 7, 9), 0)]:
        mlp = wl.xavier_mlp(dims, seed=5, act=act, bias_scale=0.3, feature_set=1 if dims[0] == 16 else 0)
        x = rng.normal(size=dims[0]).astype(np.float32) * mlp["x_scale"] + mlp["x_mean"]
        z = (x.astype(np.float64) - mlp["x_mean"]) / mlp["x_scale"].astype(np.float64)
        for l, (W, b) in enumerate(zip(mlp["W"], mlp["b"])):
            z = W.astype(np.float64) @ z + b
            if l < len(mlp["W"]) - 1:
                z = z / (1 + np.exp(-z)) if act == 0 else np.maximum(z, 0)
        ref = z * mlp["y_scale"] + mlp["y_mean"]
        np.testing.assert_allclose(orc.mlp_forward(mlp, x), ref, rtol=1e-12, atol=1e-14)
    # the head is linear: doubling the last layer's W and b doubles (y - y_mean)
    mlp = _mlp((13, 64, 64, 64, 9))
    x = rng.normal(size=13).astype(np.float32)
    y1 = orc.mlp_forward(mlp, x)
    m2 = dict(mlp)
    m2["W"] = mlp["W"][:-1] + [2 * mlp["W"][-1]]
    m2["b"] = mlp["b"][:-1] + [2 * mlp["b"][-1]]
    np.testing.assert_allclose(orc.mlp_forward(m2, x) - mlp["y_mean"], 2 * (y1 - mlp["y_mean"]), rtol=1e-13)


def test_features_and_flags(orc):
    """13-feature set (BASELINE config 1: n, u3, T, 5 traceless stress, 3 heat flux) from hand-made records."""
    mlp = wl.xavier_mlp((13, 64, 64, 64, 9), n_scale=0.01, theta_ref=0.5, tau=2.0)
    lite = np.array([200, 0.1, 0.2, 0.3, 0.6, 0.01, 0.02, 0.5, 0.03, 0.4, 0.05, -0.06, 0.07])
    th = (0.6 + 0.5 + 0.4) / 3
    x = orc.mlp_features(lite, mlp)
    ref = [2.0, 0.1, 0.2, 0.3, th / 0.5, 2 * (0.6 - th), 0.02, 0.04, 2 * (0.5 - th), 0.06, 0.05, -0.06, 0.07]
    np.testing.assert_allclose(x, np.float32(ref), rtol=1e-7)
    # the FULL record gives the same features (h_i = t_ikk)
    full = np.zeros(29)
    full[:10] = lite[:10]
    full[10], full[13], full[15] = 0.02, 0.02, 0.01          # t111 + t122 + t133 = 0.05
    full[11], full[16], full[18] = -0.01, -0.02, -0.03       # t112 + t222 + t233 = -0.06
    full[12], full[17], full[19] = 0.03, 0.03, 0.01          # t113 + t223 + t333 = 0.07
    np.testing.assert_allclose(orc.mlp_features(full, mlp), x, rtol=1e-6)
    # 16-feature set: rho, T, U, Pi = n P (6), q, DM2 = 3 theta, nu = 1/tau
    m16 = wl.xavier_mlp((16, 8, 9), feature_set=1, n_scale=0.01, tau=2.0)
    x16 = orc.mlp_features(lite, m16, tau=2.0)
    ref16 = [2.0, th / 0.5, 0.1, 0.2, 0.3, 1.2, 0.02, 0.04, 1.0, 0.06, 0.8, 0.05, -0.06, 0.07, 3 * th, 0.5]
    np.testing.assert_allclose(x16, np.float32(ref16), rtol=1e-7)
    # flags: empty -> zeros; low count / cold -> Langevin; relax_w blends with the old coefficients
    recs = np.stack([lite, np.zeros(13), np.r_[1.0, lite[1:]], np.r_[lite[:4], np.zeros(9)]])
    coef, flags = orc.closure_mlp(recs, mlp, 2.0)
    assert flags.tolist() == [0, orc.FLAG_EMPTY, orc.FLAG_LOWCOUNT, orc.FLAG_SINGULAR]
    np.testing.assert_allclose(coef[0], orc.mlp_forward(mlp, x), rtol=1e-14)
    assert np.all(coef[1] == 0) and coef[2].tolist() == [-0.5, 0, 0, -0.5, 0, -0.5, 0, 0, 0]
    old = np.full((4, 9), 7.0)
    c2, _ = orc.closure_mlp(recs, mlp, 2.0, relax_w=0.2, coef_old=old)
    np.testing.assert_allclose(c2[0], 0.2 * coef[0] + 0.8 * 7.0, rtol=1e-14)
    # ... unless the cell has no history (R12: all nine old coefficients zero, e.g. EMPTY at the previous step)
    old[0] = 0.0
    old[2] = 0.0
    old[3, 4] = 0.0                                            # one zero among nine is still a history
    c3, _ = orc.closure_mlp(recs, mlp, 2.0, relax_w=0.2, coef_old=old)
    assert np.array_equal(c3[0], coef[0]) and np.array_equal(c3[2], coef[2])
    np.testing.assert_allclose(c3[3], 0.2 * coef[3] + 0.8 * old[3], rtol=1e-14)


# ------------------------------------------------------------------------------------------------ S6
def test_philox_known_answers(orc):
    n = 0
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.strip() and not line.startswith("#"):
            w = [int(t, 16) for t in line.split()]
            assert orc.philox4x32_10(w[0:4], w[4:6]).tolist() == w[6:10]
            n += 1
    assert n == 3


def test_philox_single_round_structure(orc):
    """Brute-force re-statement with Python big integers (not C): the bijection of Salmon et al., ten rounds."""
    def philox(ctr, key):
        c, k = list(ctr), list(key)
        for _ in range(10):
            p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
            c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
            k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
        return c
    rng = np.random.default_rng(1)
    for _ in range(50):
        w = rng.integers(0, 2 ** 32, size=6, dtype=np.uint64)
        assert orc.philox4x32_10(w[:4], w[4:]).tolist() == philox([int(v) for v in w[:4]], [int(v) for v in w[4:]])


def test_uniform_mapping_and_counter_layout(orc):
    pid, step, stream, seed = 12345, (7 << 32) | 99, 2, (0xDEADBEEF << 32) | 0x1234
    w = orc.philox4x32_10([pid, 99, 7, 2], [0x1234, 0xDEADBEEF])
    u = orc.uniforms(pid, step, stream, seed)[0]
    expect = ((w >> 9).astype(np.float64) + 0.5) / 2 ** 23
    assert np.array_equal(u, expect)
    assert np.array_equal(u.astype(np.float32).astype(np.float64), u)        # exact in fp32, in (0,1)
    assert np.all((u > 0) & (u < 1))
    xi = orc.normals(pid, step, stream, seed)[0]
    r0, r1 = math.sqrt(-2 * math.log(u[0])), math.sqrt(-2 * math.log(u[2]))
    np.testing.assert_allclose(xi, [r0 * math.cos(2 * math.pi * u[1]), r0 * math.sin(2 * math.pi * u[1]),
                                    r1 * math.cos(2 * math.pi * u[3])], rtol=1e-14, atol=1e-15)


def test_normal_statistics(orc):
    xi = orc.normals(np.arange(200_000, dtype=np.uint32), 3, 0, 42)
    n = xi.size
    assert np.max(np.abs(xi.mean(0))) < 5 / math.sqrt(n / 3)
    assert np.max(np.abs(xi.var(0) - 1)) < 5 * math.sqrt(2 / (n / 3))
    kurt = (xi ** 4).mean()
    assert abs(kurt - 3) < 5 * math.sqrt(96 / n)
    assert np.max(np.abs(xi)) <= math.sqrt(-2 * math.log(2 ** -24)) + 1e-12       # = 5.768...
    assert abs(np.corrcoef(xi.T)[0, 1]) < 0.01 and abs(np.corrcoef(xi.T)[0, 2]) < 0.01
    # a different step or stream gives a different, uncorrelated draw
    other = orc.normals(np.arange(20_000, dtype=np.uint32), 4, 0, 42)
    assert abs(np.corrcoef(xi[:20_000, 0], other[:, 0])[0, 1]) < 0.03
