"""Seeded synthetic workloads shaped like the paper's runs.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.  It holds none of the method's
arithmetic (no moments, closure, Philox, update): it only draws particle ensembles with numpy's own generators
and writes down configuration numbers.  numpy only -- no torch, no native code -- so it imports anywhere.

Units: velocities in c_mp = sqrt(2 k T_ref / m) (argon), so theta_ref = 0.5; lengths in L
(Couette, cavity) or cells (cylinder); time in L / c_mp.  Relaxation time from Kn (reading):
tau = 2 sqrt(pi) Kn L / c_mp.

The paper's own particle data, Supplementary Table S1 and trained weights are not available; these inputs stand
in for its Couette (:278-282), cavity (:380-396) and hypersonic-cylinder (:545, :668) runs.
"""
import math

import numpy as np

THETA_REF = 0.5
WALL_NONE, WALL_DIFFUSE, WALL_PERIODIC, WALL_INFLOW = 0, 1, 2, 3


def tau_from_kn(kn, L=1.0):
    return 2.0 * math.sqrt(math.pi) * kn * L


def _rng(seed):
    return np.random.Generator(np.random.Philox(seed))


def make_config(nx, ny, dx, dy, dt, tau, walls, x0=0.0, y0=0.0, eps2_scale=1.0, min_count=10, conserve_mode=1,
                seed=0, body=None, max_particles=0):
    """Plain dict understood by both sides.  walls: 4 x (kind, theta_w, ux, uy, uz) for xmin, xmax, ymin, ymax."""
    f = lambda v: float(np.float32(v))  # noqa: E731  (every float is an fp32 value on both sides)
    return dict(nx=int(nx), ny=int(ny), x0=f(x0), y0=f(y0), dx=f(dx), dy=f(dy), dt=f(dt), tau=f(tau),
                eps2_scale=f(eps2_scale), min_count=int(min_count), min_count_mlp=2,
                conserve_mode=int(conserve_mode), seed=int(seed),
                walls=[(int(w[0]),) + tuple(f(v) for v in w[1:]) for w in walls],
                body=None if body is None else tuple(f(v) for v in body), max_particles=int(max_particles))


NO_WALLS = [(WALL_NONE, 0.5, 0, 0, 0)] * 4


def _positions_in_cells(rng, counts, nx, ny, dx, dy, x0=0.0, y0=0.0):
    """Uniform positions inside each cell; counts[ncell] particles per cell (cell = iy*nx + ix)."""
    cell = np.repeat(np.arange(nx * ny), counts)
    ix, iy = cell % nx, cell // nx
    n = cell.shape[0]
    # keep a margin so that fp32 rounding cannot move a particle out of its cell
    u = rng.uniform(0.001, 0.999, size=(2, n))
    x = (x0 + (ix + u[0]) * dx).astype(np.float32)
    y = (y0 + (iy + u[1]) * dy).astype(np.float32)
    return x, y, cell


def _finish(rng, x, y, v, shuffle):
    n = x.shape[0]
    state = dict(x=x, y=y, vx=v[:, 0].astype(np.float32), vy=v[:, 1].astype(np.float32),
                 vz=v[:, 2].astype(np.float32))
    if shuffle:
        p = rng.permutation(n)
        state = {k: np.ascontiguousarray(a[p]) for k, a in state.items()}
    else:
        state = {k: np.ascontiguousarray(a) for k, a in state.items()}
    state["pid"] = np.arange(n, dtype=np.uint32)
    return state


# ------------------------------------------------------------------------------------------------ C1
def couette(nx=50, ppc=100, kn=0.15, seed=0, shuffle=True):
    """BASELINE config 1: 1D Couette, 50 cells x 100 ppc, Maxwellian + linear shear +-0.3."""
    rng = _rng(seed)
    dx = 1.0 / nx
    tau = tau_from_kn(kn)
    walls = [(WALL_DIFFUSE, THETA_REF, 0, -0.3, 0), (WALL_DIFFUSE, THETA_REF, 0, 0.3, 0),
             (WALL_NONE, THETA_REF, 0, 0, 0), (WALL_NONE, THETA_REF, 0, 0, 0)]
    cfg = make_config(nx, 1, dx, 1.0, 0.1 * tau, tau, walls, seed=seed, max_particles=nx * ppc)
    counts = np.full(nx, ppc)
    x, y, _ = _positions_in_cells(rng, counts, nx, 1, dx, 1.0)
    v = rng.normal(0.0, math.sqrt(THETA_REF), size=(x.shape[0], 3))
    v[:, 1] += 0.3 * (2.0 * x - 1.0)
    return cfg, _finish(rng, x, y, v, shuffle)


# ------------------------------------------------------------------------------------------------ C2
def grad13_cells(ncx=100, ncy=100, ppc=50, seed=1, shuffle=False, smax=0.3, qmax=0.2, bulk=0.3):
    """BASELINE config 2: per-cell Grad-13-perturbed Maxwellians by acceptance-rejection (no streaming).
    Returns cfg, state (cell-sorted unless shuffle) and the per-cell (s, qhat, bulk) that were drawn."""
    rng = _rng(seed)
    nc = ncx * ncy
    dx, dy = 1.0 / ncx, 1.0 / ncy
    cfg = make_config(ncx, ncy, dx, dy, 0.1, 1.0, NO_WALLS, seed=seed, max_particles=nc * ppc)
    # symmetric traceless s with max |s_ij| <= smax
    a = rng.uniform(-1, 1, size=(nc, 3, 3))
    s = 0.5 * (a + a.transpose(0, 2, 1))
    s -= np.eye(3) * (np.trace(s, axis1=1, axis2=2) / 3.0)[:, None, None]
    s *= (smax * rng.uniform(0.2, 1.0, size=nc) / np.abs(s).reshape(nc, 9).max(axis=1))[:, None, None]
    # qhat uniform in the ball |q| <= qmax
    d = rng.normal(size=(nc, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    qh = d * (qmax * rng.uniform(0, 1, size=nc) ** (1.0 / 3.0))[:, None]
    out = np.empty((nc, ppc, 3))
    need = np.full(nc, ppc)
    wmax = 4.0
    while need.max() > 0:
        idx = np.nonzero(need > 0)[0]
        m = 4 * ppc
        Cc = rng.normal(0.0, math.sqrt(0.5), size=(idx.shape[0], m, 3))  # C = c / c_mp
        C2 = (Cc ** 2).sum(-1)
        w = 1.0 + np.einsum("nij,nmi,nmj->nm", s[idx], Cc, Cc) + 0.8 * np.einsum("ni,nmi->nm", qh[idx], Cc) * (C2 - 2.5)
        acc = rng.uniform(0, wmax, size=w.shape) < w  # negative weights never accepted
        for r, c in enumerate(idx):
            got = Cc[r][acc[r]][: need[c]]
            k = ppc - need[c]
            out[c, k:k + got.shape[0]] = got
            need[c] -= got.shape[0]
    ub = rng.uniform(-bulk, bulk, size=(nc, 3))
    v = (out + ub[:, None, :]).reshape(nc * ppc, 3)
    x, y, _ = _positions_in_cells(rng, np.full(nc, ppc), ncx, ncy, dx, dy)
    return cfg, _finish(rng, x, y, v, shuffle), dict(s=s, qhat=qh, bulk=ub)


# ------------------------------------------------------------------------------------------------ C3 / C4
def cavity(n=200, ppc=100, kn=0.5, seed=3, shuffle=True, lid=0.148):
    """BASELINE configs 3/4: 2D lid-driven cavity, n x n cells, diffuse isothermal walls, lid (ymax) moving in x
    at 50 m/s = 0.148 c_mp.  dt = min(0.1 tau, 0.5 dx) (reading; the paper gives no dt rule)."""
    rng = _rng(seed)
    dx = 1.0 / n
    tau = tau_from_kn(kn)
    dt = min(0.1 * tau, 0.5 * dx)
    walls = [(WALL_DIFFUSE, THETA_REF, 0, 0, 0), (WALL_DIFFUSE, THETA_REF, 0, 0, 0),
             (WALL_DIFFUSE, THETA_REF, 0, 0, 0), (WALL_DIFFUSE, THETA_REF, lid, 0, 0)]
    cfg = make_config(n, n, dx, dx, dt, tau, walls, seed=seed, max_particles=n * n * ppc)
    x, y, _ = _positions_in_cells(rng, np.full(n * n, ppc), n, n, dx, dx)
    v = rng.normal(0.0, math.sqrt(THETA_REF), size=(x.shape[0], 3)).astype(np.float32)
    return cfg, _finish(rng, x, y, v, shuffle)


# ------------------------------------------------------------------------------------------------ C5
def cylinder_field(nx=400, ny=300, ppc_inf=100.0):
    """Analytic bow-shock-like field on an nx x ny grid (lengths in cells).  Returns per-cell rho, theta, U (2 comps),
    inside-body mask and the shock-band mask.  Shapes follow SURVEY.md 8(d) C5; numbers from PAPER.md:545."""
    sx, sy = nx / 400.0, ny / 300.0
    cx, cy, R = 150.0 * sx, 150.0 * sy, 30.0 * sx
    ix, iy = np.meshgrid(np.arange(nx) + 0.5, np.arange(ny) + 0.5)  # [ny, nx]
    X, Y = ix, iy
    yy = (Y - cy) / sx
    xs = (108.0 + yy ** 2 / 120.0) * sx                     # shock surface x_s(y)
    r = np.hypot(X - cx, Y - cy)
    inside = r < R
    xb = np.where(np.abs(Y - cy) < R, cx - np.sqrt(np.maximum(R * R - (Y - cy) ** 2, 0.0)), cx)
    down = X >= xs
    xi = np.clip((X - xs) / np.maximum(xb - xs, 1.0), 0.0, 1.0)        # 0 at the shock, 1 at the body / x = cx
    wy = np.exp(-((Y - cy) / (2.0 * R)) ** 2)                          # strength falls away from the axis
    rho = np.ones_like(X)
    theta = np.full_like(X, 0.5)
    ux = np.full_like(X, 9.09)
    uy = np.zeros_like(X)
    rho_d = 1.0 + (3.883 - 1.0) * (0.35 + 0.65 * wy) + (8.0 - 3.883) * wy * xi ** 2
    th_post = 0.5 + (16.06 - 0.5) * (0.15 + 0.85 * wy)
    near = np.clip((r - R) / (0.25 * R), 0.0, 1.0)                     # thermal layer on the wall
    th_d = 1.25 + (th_post - 1.25) * near
    ux_d = 9.09 * (0.26 + 0.5 * (1 - wy)) * np.clip((r - R) / (1.5 * R), 0.0, 1.0)
    uy_d = 9.09 * 0.25 * np.sign(Y - cy) * (1 - wy) * np.clip((r - R) / R, 0, 1)
    rear = X > cx                                                       # expansion behind the shoulder
    fall = np.exp(-np.clip((X - cx) / (4.0 * R), 0, None))
    rho_d = np.where(rear, 1.0 + (rho_d - 1.0) * fall, rho_d)
    th_d = np.where(rear, 0.5 + (th_d - 0.5) * fall, th_d)
    wake = rear & (np.abs(Y - cy) < R)
    rho_d = np.where(wake, 0.05 + 0.15 * np.clip((X - cx - R) / (6 * R), 0, 1), rho_d)
    th_d = np.where(wake, 2.0, th_d)
    ux_d = np.where(wake, 0.5, ux_d)
    rho = np.where(down, rho_d, rho)
    theta = np.where(down, th_d, theta)
    ux = np.where(down, ux_d, ux)
    uy = np.where(down, uy_d, uy)
    band = np.abs(X - xs) < 3.0 * sx
    ppc = np.clip(np.rint(ppc_inf * rho), 5, 400).astype(np.int64)
    ppc[inside] = 0
    return dict(rho=rho, theta=theta, ux=ux, uy=uy, inside=inside, band=band, ppc=ppc, cx=cx, cy=cy, R=R,
                th_post=th_post, rho_post=rho_d)


def cylinder(nx=400, ny=300, seed=5, target=20_000_000, shuffle=False, kn_inf=0.01):
    """BASELINE config 5: hypersonic cylinder-like ensemble with 5..400 particles per cell (~20M at full size).
    Returns cfg, state and tau_cell (fp32, tau_inf * ppc_inf / N, tau ~ 1/n)."""
    rng = _rng(seed)
    ppc_inf = 100.0
    for _ in range(8):                                   # tune ppc_inf so that the total is close to target
        f = cylinder_field(nx, ny, ppc_inf)
        tot = int(f["ppc"].sum())
        if abs(tot - target) <= 0.02 * target:
            break
        ppc_inf *= target / tot
    counts = f["ppc"].reshape(-1)
    D = 2.0 * f["R"]
    tau_inf = tau_from_kn(kn_inf, D) / math.sqrt(2 * THETA_REF)   # c_mp = 1 at the freestream temperature
    # outer faces: freestream reservoir (a particle that leaves re-enters at xmin from the Mach-10 freestream; reading R11)
    walls = [(WALL_INFLOW, THETA_REF, 9.09, 0, 0)] * 4
    cfg = make_config(nx, ny, 1.0, 1.0, 0.055, tau_inf, walls, seed=seed, body=(f["cx"], f["cy"], f["R"], 1.25),
                      max_particles=int(counts.sum()))
    x, y, cell = _positions_in_cells(rng, counts, nx, ny, 1.0, 1.0)
    n = x.shape[0]
    th = f["theta"].reshape(-1)[cell]
    U = np.stack([f["ux"].reshape(-1)[cell], f["uy"].reshape(-1)[cell], np.zeros(n)], axis=1)
    # two-Maxwellian mixture in the shock band: a particle is upstream-like with probability 1/2
    band = f["band"].reshape(-1)[cell] & (rng.uniform(size=n) < 0.5)
    th = np.where(band, 0.5, th)
    U[band] = (9.09, 0.0, 0.0)
    v = (U + rng.normal(size=(n, 3)) * np.sqrt(th)[:, None]).astype(np.float32)
    with np.errstate(divide="ignore"):
        tau_cell = np.where(counts > 0, tau_inf * ppc_inf / np.maximum(counts, 1), tau_inf).astype(np.float32)
    cfg["ppc_inf"] = float(ppc_inf)
    return cfg, _finish(rng, x, y, v, shuffle), tau_cell


# ------------------------------------------------------------------------------------------------ MLP weights
def xavier_mlp(dims=(13, 64, 64, 64, 9), seed=0, act=0, feature_set=0, n_scale=0.01, theta_ref=THETA_REF, tau=1.0,
               bias_scale=0.0):
    """Xavier-uniform weights U(-a, a), a = sqrt(6/(fan_in+fan_out)) (BASELINE.json config 1: 'Xavier weights from
    seed 0'), zero biases unless bias_scale > 0.  Input standardisation is set to nominal values of the features;
    outputs are centred on the Langevin coefficients (c = -delta/tau, gamma = 0) with a spread of 0.1/tau, so the
    random network is a perturbation of the linear model.  No trained weights exist in this container."""
    rng = _rng(seed)
    dims = [int(d) for d in dims]
    W, b = [], []
    for l in range(len(dims) - 1):
        a = math.sqrt(6.0 / (dims[l] + dims[l + 1]))
        W.append(rng.uniform(-a, a, size=(dims[l + 1], dims[l])).astype(np.float32))
        b.append((bias_scale * rng.uniform(-1, 1, size=dims[l + 1])).astype(np.float32))
    if feature_set == 0:
        x_mean = [1.0, 0, 0, 0, 1.0] + [0.0] * 8
        x_scale = [0.1, 0.3, 0.3, 0.3, 0.15] + [0.05] * 5 + [0.05] * 3
    else:
        x_mean = [1.0, 1.0, 0, 0, 0, 0.5, 0, 0, 0.5, 0, 0.5, 0, 0, 0, 1.5, 1.0 / tau]
        x_scale = [0.1, 0.15, 0.3, 0.3, 0.3] + [0.05] * 6 + [0.05] * 3 + [0.2, 0.1 / tau]
    assert len(x_mean) == dims[0] and len(x_scale) == dims[0]
    y_mean = np.array([-1 / tau, 0, 0, -1 / tau, 0, -1 / tau, 0, 0, 0], dtype=np.float32)
    y_scale = np.array([0.1 / tau] * 6 + [0.1 / (tau * math.sqrt(theta_ref))] * 3, dtype=np.float32)
    return dict(dims=np.array(dims, dtype=np.int32), W=W, b=b, x_mean=np.array(x_mean, dtype=np.float32),
                x_scale=np.array(x_scale, dtype=np.float32), y_mean=y_mean, y_scale=y_scale, act=int(act),
                feature_set=int(feature_set), n_scale=float(np.float32(n_scale)),
                theta_ref=float(np.float32(theta_ref)))


# ------------------------------------------------------------------------------------------------ ragged test case
def ragged(nx=37, ny=23, seed=7, mean_ppc=40.0, empty_frac=0.1, shuffle=True, walls=None, drift=0.0):
    """Edge-case ensemble for parity tests: per-cell counts 0..~4x mean (about ``empty_frac`` empty cells, some
    cells with 1-3 particles, a few very full ones), per-cell bulk velocity (+ ``drift`` on x) and temperature."""
    rng = _rng(seed)
    nc = nx * ny
    dx, dy = 1.0 / nx, 1.0 / ny
    lam = mean_ppc * rng.gamma(2.0, 0.5, size=nc)
    counts = rng.poisson(lam)
    counts[rng.uniform(size=nc) < empty_frac] = 0
    small = rng.uniform(size=nc) < 0.05
    counts[small] = rng.integers(1, 4, size=int(small.sum()))
    big = rng.integers(0, nc, size=3)
    counts[big] = (mean_ppc * rng.integers(8, 14, size=3)).astype(np.int64)
    cfg = make_config(nx, ny, dx, dy, 0.02, 0.7, walls or NO_WALLS, seed=seed, max_particles=int(counts.sum()))
    x, y, cell = _positions_in_cells(rng, counts, nx, ny, dx, dy)
    n = x.shape[0]
    th = rng.uniform(0.2, 1.5, size=nc)[cell]
    U = rng.uniform(-0.5, 0.5, size=(nc, 3))[cell]
    U[:, 0] += drift
    v = U + rng.normal(size=(n, 3)) * np.sqrt(th)[:, None]
    # skew the distribution a little so that odd moments are not pure noise
    v += 0.15 * (rng.exponential(size=(n, 3)) - 1.0) * np.sqrt(th)[:, None]
    return cfg, _finish(rng, x, y, v, shuffle)
