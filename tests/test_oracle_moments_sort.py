"""Pins for the oracle's S1 (cell index / stable sort) and S0 (moments).  CPU only.

Each pin is something other than the oracle itself: hand values (tests/golden/moments_hand.txt), closed forms of a
Maxwellian (PAPER.md:415: Delta4 = <c^4> - 15 theta^2 -> 0; :651: D_G = -1/2 log det(P/theta) -> 0), Galilean
invariance, axis-permutation symmetry, numpy's stable argsort, invariants of a permutation.
"""
import os

import numpy as np
import pytest

from paper_2606_15622_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")

FULL = ["N", "U1", "U2", "U3", "P11", "P12", "P13", "P22", "P23", "P33",
        "t111", "t112", "t113", "t122", "t123", "t133", "t222", "t223", "t233", "t333",
        "F11", "F12", "F13", "F22", "F23", "F33", "g1", "g2", "g3"]
LITE = FULL[:10] + ["h1", "h2", "h3"]


def _one_cell(orc, v, mode):
    v = np.asarray(v, dtype=np.float32)
    cs = np.array([0, v.shape[0]], dtype=np.int32)
    return orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, mode)[0]


def test_hand_values(orc):
    gold = {}
    for line in open(os.path.join(GOLD, "moments_hand.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            gold[k] = float(v)
    sets = {"A": [(1, 0, 0), (-1, 0, 0), (0, 2, 0), (0, -2, 0)], "B": [(0, 0, 0), (0, 0, 0), (3, 0, 0)]}
    for name, v in sets.items():
        m = dict(zip(FULL, _one_cell(orc, v, 1)))
        for k, val in gold.items():
            case, key = k.split(".")
            if case == name:
                assert m[key] == pytest.approx(val, abs=1e-14), k
    # case A: everything not listed that is odd in any component vanishes, and theta = 5/6
    mA = dict(zip(FULL, _one_cell(orc, sets["A"], 1)))
    assert (mA["P11"] + mA["P22"] + mA["P33"]) / 3 == pytest.approx(5 / 6, abs=1e-15)
    for k in ["P12", "P13", "P23"] + FULL[10:20] + ["F12", "F13", "F23", "g2", "g3"]:
        assert mA[k] == 0.0
    # case B: h1 = t111 + t122 + t133 = 2 and F = F11 = 6
    lite = dict(zip(LITE, _one_cell(orc, sets["B"], 0)))
    assert lite["h1"] == pytest.approx(2.0, abs=1e-14) and lite["h2"] == 0 and lite["h3"] == 0


def test_lite_is_contraction_of_full(orc):
    rng = np.random.default_rng(7)
    v = rng.normal(size=(257, 3)) * [0.5, 1.0, 2.0] + [3, -2, 1]
    f = dict(zip(FULL, _one_cell(orc, v, 1)))
    l = dict(zip(LITE, _one_cell(orc, v, 0)))
    for k in FULL[:10]:
        assert l[k] == f[k]
    assert l["h1"] == pytest.approx(f["t111"] + f["t122"] + f["t133"], rel=1e-13)
    assert l["h2"] == pytest.approx(f["t112"] + f["t222"] + f["t233"], rel=1e-13)
    assert l["h3"] == pytest.approx(f["t113"] + f["t223"] + f["t333"], rel=1e-13)


def test_maxwellian_closed_forms(orc):
    """P -> theta I, t -> 0, F_ij -> 5 theta^2 delta_ij, F -> 15 theta^2, g -> 0 within 5 standard errors."""
    n, theta = 1_000_000, 0.5
    rng = np.random.default_rng(11)
    v = rng.normal(0.0, np.sqrt(theta), size=(n, 3)) + [0.3, -0.2, 0.1]
    m = dict(zip(FULL, _one_cell(orc, v, 1)))
    se = 5.0 / np.sqrt(n)
    s = np.sqrt(theta)
    assert m["N"] == n
    for k, u in zip(("U1", "U2", "U3"), np.float32([0.3, -0.2, 0.1])):
        assert abs(m[k] - u) < se * s
    # Gaussian moments: var(c_i c_j)=theta^2 (i!=j), var(c_i^2)=2 theta^2; bounds below are loose multiples
    for k in ("P11", "P22", "P33"):
        assert abs(m[k] - theta) < se * 2 * theta
    for k in ("P12", "P13", "P23"):
        assert abs(m[k]) < se * theta
    for k in FULL[10:20]:
        assert abs(m[k]) < se * 4 * s ** 3           # sd of c^3-type products <= sqrt(15) theta^1.5
    for k in ("F11", "F22", "F33"):
        assert abs(m[k] - 5 * theta ** 2) < se * 30 * theta ** 2
    for k in ("F12", "F13", "F23"):
        assert abs(m[k]) < se * 12 * theta ** 2
    F = m["F11"] + m["F22"] + m["F33"]
    assert abs(F - 15 * theta ** 2) < se * 60 * theta ** 2          # Delta4 -> 0
    for k in ("g1", "g2", "g3"):
        assert abs(m[k]) < se * 120 * s ** 5
    P = np.array([[m["P11"], m["P12"], m["P13"]], [m["P12"], m["P22"], m["P23"]], [m["P13"], m["P23"], m["P33"]]])
    th = np.trace(P) / 3
    DG = -0.5 * np.log(np.linalg.det(P / th))                       # PAPER.md:651, D_G >= 0, -> 0 at equilibrium
    assert 0 <= DG < 1e-4


def test_galilean_invariance_mach10(orc):
    """Adding the paper's U_inf = 2624 to every velocity leaves all central moments unchanged.
    Velocities are multiples of 2^-12 so that v + 2624 is exact in fp32 and both ensembles are identical."""
    rng = np.random.default_rng(5)
    v = np.round(rng.normal(0, 290.0, size=(400, 3)) * 4096) / 4096
    assert np.all(np.abs(v) < 2048)
    a = _one_cell(orc, v, 1)
    shifted = (v + [2624.0, 0, 0]).astype(np.float32)
    assert np.array_equal(shifted.astype(np.float64), v + [2624.0, 0, 0])
    b = _one_cell(orc, shifted, 1)
    assert b[1] - a[1] == pytest.approx(2624.0, abs=1e-9)
    scale = np.array([290.0 ** k for k in [2] * 6 + [3] * 10 + [4] * 6 + [5] * 3])
    assert np.max(np.abs(b[4:] - a[4:]) / scale) < 1e-12


def test_axis_permutation(orc):
    rng = np.random.default_rng(3)
    v = rng.normal(size=(300, 3)) ** 3
    a = dict(zip(FULL, _one_cell(orc, v, 1)))
    b = dict(zip(FULL, _one_cell(orc, v[:, [1, 2, 0]], 1)))   # new axis 1 = old 2, new 2 = old 3, new 3 = old 1
    old = {1: 2, 2: 3, 3: 1}

    def ren(name):
        head, idx = name[0], name[1:]
        return head + "".join(sorted(str(old[int(ch)]) for ch in idx))
    for k in FULL[1:]:
        assert b[k] == pytest.approx(a[ren(k)], rel=1e-12, abs=1e-13), k


def test_empty_and_ragged_cells(orc):
    v = np.arange(30, dtype=np.float32).reshape(10, 3)
    cs = np.array([0, 0, 1, 1, 10], dtype=np.int32)         # empty, single particle, empty, nine
    m = orc.cell_moments(v[:, 0], v[:, 1], v[:, 2], cs, 1)
    assert np.all(m[0] == 0) and np.all(m[2] == 0)
    assert m[1, 0] == 1 and np.array_equal(m[1, 1:4], v[0]) and np.all(m[1, 4:] == 0)
    assert m[3, 0] == 9


# ------------------------------------------------------------------------------------------------ S1
def test_cell_index_matches_fp32_numpy(orc):
    cfg, st = wl.cavity(16, 7, seed=9)
    x = st["x"].copy()
    x[:5] = [-0.5, 1.5, np.nan, 0.0, np.nextafter(np.float32(1.0), np.float32(0))]
    key = orc.cell_index(x, st["y"], cfg)
    inv_dx = np.float32(1.0) / np.float32(cfg["dx"])
    fx = np.floor((x - np.float32(cfg["x0"])) * inv_dx)
    ix = np.where(np.isnan(fx) | (fx < 0), 0, np.minimum(fx, cfg["nx"] - 1)).astype(np.int64)
    fy = np.floor((st["y"] - np.float32(cfg["y0"])) * (np.float32(1.0) / np.float32(cfg["dy"])))
    iy = np.clip(fy, 0, cfg["ny"] - 1).astype(np.int64)
    assert np.array_equal(key, iy * cfg["nx"] + ix)
    assert key[:5].tolist() == [int(iy[0]) * 16 + 0, int(iy[1]) * 16 + 15, int(iy[2]) * 16 + 0, int(iy[3]) * 16, int(iy[4]) * 16 + 15]


def test_stable_sort_against_numpy_and_invariants(orc):
    rng = np.random.default_rng(2)
    for n, ncell in [(0, 5), (1, 1), (1000, 7), (5000, 5000), (20000, 300)]:
        key = rng.integers(0, ncell, size=n).astype(np.int32)
        cs, perm = orc.sort_by_key(key, ncell)
        assert np.array_equal(perm, np.argsort(key, kind="stable").astype(np.uint32))
        assert np.array_equal(np.sort(perm), np.arange(n, dtype=np.uint32))
        assert np.all(np.diff(key[perm]) >= 0)
        assert cs[0] == 0 and cs[-1] == n and np.all(np.diff(cs) >= 0)
        assert np.array_equal(np.diff(cs), np.bincount(key, minlength=ncell))


def test_sort_by_cell_counts_match_generator(orc):
    cfg, st = wl.cavity(12, 9, seed=4)
    out, cs, perm = orc.sort_by_cell(st, cfg)
    assert np.all(np.diff(cs) == 9)                       # generator puts exactly ppc particles in every cell
    for k in ("x", "vx", "pid"):
        assert np.array_equal(out[k], st[k][perm])
