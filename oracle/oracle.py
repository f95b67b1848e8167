"""ctypes/numpy marshalling for ``fp_oracle.c`` (see the header of that file; TEST INFRASTRUCTURE ONLY).

No arithmetic of the method lives here except the composition of one step (``step``), which only orders calls.
A configuration is a plain ``dict`` (keys: nx, ny, x0, y0, dx, dy, dt, tau, eps2_scale, min_count,
conserve_mode, seed, walls = 4 x (kind, theta_w, ux, uy, uz), body = None | (cx, cy, R, theta_w)).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fp_oracle.c")
_LIB = os.path.join(_HERE, "libfp_oracle.so")

FLAG_EMPTY, FLAG_LOWCOUNT, FLAG_SINGULAR, FLAG_ILLCOND, FLAG_ALPHA, FLAG_SKIPPED, FLAG_NONFINITE = 1, 2, 4, 8, 16, 32, 64

_lib = None


def build(force=False):
    """Compile fp_oracle.c with gcc (-O2 -ffp-contract=off so fp32 position arithmetic is not fused).
    ORACLE_SANITIZE=1 in the environment builds and loads an AddressSanitizer + UndefinedBehaviorSanitizer variant instead
    (run the CPU pins with LD_PRELOAD=$(gcc -print-file-name=libasan.so); summary under profiles/)."""
    global _LIB
    san = os.environ.get("ORACLE_SANITIZE") == "1"
    if san:
        _LIB = os.path.join(_HERE, "libfp_oracle_asan.so")
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        extra = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-g", "-O1"] if san else ["-O2"]
        subprocess.check_call(["gcc"] + extra + ["-ffp-contract=off", "-fno-fast-math", "-std=c11", "-fopenmp", "-shared",
                               "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _u32(a):
    return np.ascontiguousarray(a, dtype=np.uint32)


def set_threads(n=0):
    """Threads of the per-cell / per-particle loops (0 = all cores).  Results do not depend on it."""
    lib().orc_set_threads(C.c_int(int(n)))
    return int(lib().orc_max_threads())


def ncell_of(cfg):
    return int(cfg["nx"]) * int(cfg["ny"])


# ---------------------------------------------------------------- S1
def cell_index(x, y, cfg):
    x, y = _f32(x), _f32(y)
    key = np.empty(x.shape[0], dtype=np.int32)
    lib().orc_cell_index(C.c_int64(x.shape[0]), _p(x, C.c_float), _p(y, C.c_float), C.c_int32(cfg["nx"]),
                         C.c_int32(cfg["ny"]), C.c_float(cfg["x0"]), C.c_float(cfg["y0"]), C.c_float(cfg["dx"]),
                         C.c_float(cfg["dy"]), _p(key, C.c_int32))
    return key


def sort_by_key(key, ncell):
    key = _i32(key)
    cell_start = np.empty(ncell + 1, dtype=np.int32)
    perm = np.empty(key.shape[0], dtype=np.uint32)
    lib().orc_sort_by_key(C.c_int64(key.shape[0]), _p(key, C.c_int32), C.c_int32(ncell), _p(cell_start, C.c_int32),
                          _p(perm, C.c_uint32))
    return cell_start, perm


def sort_by_cell(state, cfg):
    """state: dict of x,y,vx,vy,vz (f32) and pid (u32).  Returns (sorted state, cell_start, perm)."""
    key = cell_index(state["x"], state["y"], cfg)
    cell_start, perm = sort_by_key(key, ncell_of(cfg))
    out = {k: np.ascontiguousarray(state[k][perm]) for k in ("x", "y", "vx", "vy", "vz", "pid")}
    return out, cell_start, perm


# ---------------------------------------------------------------- S0
def cell_moments(vx, vy, vz, cell_start, mode):
    vx, vy, vz, cell_start = _f32(vx), _f32(vy), _f32(vz), _i32(cell_start)
    ncell = cell_start.shape[0] - 1
    mom = np.empty((ncell, 29 if mode else 13), dtype=np.float64)
    lib().orc_cell_moments(_p(vx, C.c_float), _p(vy, C.c_float), _p(vz, C.c_float), _p(cell_start, C.c_int32),
                           C.c_int32(ncell), C.c_int32(mode), _p(mom, C.c_double))
    return mom


def cell_diagnostics(mom_full, theta_inf=0.5, n_inf=1.0, dg_inf=0.0):
    """NEXT-2: 16 diagnostics per cell from the FULL record (fp_oracle.c orc_cell_diagnostics)."""
    mom_full = _f64(mom_full)
    ncell = mom_full.shape[0]
    assert mom_full.shape[1] == 29
    diag = np.empty((ncell, 16), dtype=np.float64)
    lib().orc_cell_diagnostics(C.c_int32(ncell), _p(mom_full, C.c_double), C.c_double(theta_inf), C.c_double(n_inf),
                               C.c_double(dg_inf), _p(diag, C.c_double))
    return diag


def cell_dm6(vx, vy, vz, cell_start):
    """NEXT-2: DM6 = <(c^2)^3> per cell."""
    vx, vy, vz, cell_start = _f32(vx), _f32(vy), _f32(vz), _i32(cell_start)
    ncell = cell_start.shape[0] - 1
    dm6 = np.empty(ncell, dtype=np.float64)
    lib().orc_cell_dm6(_p(vx, C.c_float), _p(vy, C.c_float), _p(vz, C.c_float), _p(cell_start, C.c_int32),
                       C.c_int32(ncell), _p(dm6, C.c_double))
    return dm6


def average_results(x, k, avg):
    """NEXT-2: running mean, in place on avg."""
    x = _f64(x)
    assert avg.dtype == np.float64 and avg.flags["C_CONTIGUOUS"] and avg.size == x.size
    lib().orc_average_results(C.c_int64(x.size), _p(x, C.c_double), C.c_int64(k), _p(avg, C.c_double))
    return avg


# ---------------------------------------------------------------- S2/S3
def _tau_args(tau, ncell):
    if np.ndim(tau) == 0:
        return None, C.POINTER(C.c_float)(), float(tau)
    t = _f32(tau)
    assert t.shape[0] == ncell
    return t, _p(t, C.c_float), 0.0


def closure_exact(mom_full, tau, eps2_scale=1.0, min_count=10):
    mom_full = _f64(mom_full)
    ncell = mom_full.shape[0]
    assert mom_full.shape[1] == 29
    keep, tau_p, tau_s = _tau_args(tau, ncell)
    coef = np.empty((ncell, 9), dtype=np.float64)
    flags = np.zeros(ncell, dtype=np.uint32)
    kappa = np.zeros(ncell, dtype=np.float64)
    lib().orc_closure_exact(C.c_int32(ncell), _p(mom_full, C.c_double), tau_p, C.c_double(tau_s),
                            C.c_double(eps2_scale), C.c_int32(min_count), _p(coef, C.c_double),
                            _p(flags, C.c_uint32), _p(kappa, C.c_double))
    return coef, flags, kappa


def closure_exact_system(m, tau, eps2_scale=1.0, min_count=10):
    """One cell: returns coef, flag, kappa and the SCALED system (A, b) the oracle assembled."""
    m = _f64(m)
    coef = np.empty(9)
    A = np.zeros((9, 9))
    b = np.zeros(9)
    flag = C.c_uint32(0)
    kappa = C.c_double(0)
    lib().orc_closure_exact_cell(_p(m, C.c_double), C.c_double(tau), C.c_double(eps2_scale), C.c_int32(min_count),
                                 _p(coef, C.c_double), C.byref(flag), C.byref(kappa), _p(A, C.c_double),
                                 _p(b, C.c_double))
    return coef, flag.value, kappa.value, A, b


# ---------------------------------------------------------------- S4
def _mlp_args(mlp):
    dims = _i32(mlp["dims"])
    nl = dims.shape[0] - 1
    Ws = [_f32(w) for w in mlp["W"]]
    bs = [_f32(b) for b in mlp["b"]]
    for l in range(nl):
        assert Ws[l].shape == (dims[l + 1], dims[l]) and bs[l].shape == (dims[l + 1],)
    Wp = (C.POINTER(C.c_float) * nl)(*[_p(w, C.c_float) for w in Ws])
    bp = (C.POINTER(C.c_float) * nl)(*[_p(b, C.c_float) for b in bs])
    sc = [_f32(mlp[k]) for k in ("x_mean", "x_scale", "y_mean", "y_scale")]
    return nl, dims, Ws, bs, Wp, bp, sc


def mlp_features(m, mlp, tau=1.0):
    m = _f64(m)
    x = np.zeros(16, dtype=np.float32)
    lib().orc_mlp_features.restype = C.c_int32
    n = lib().orc_mlp_features(_p(m, C.c_double), C.c_int32(m.shape[0]), C.c_int32(mlp.get("feature_set", 0)),
                               C.c_double(mlp.get("n_scale", 1.0)), C.c_double(mlp.get("theta_ref", 0.5)),
                               C.c_double(tau), _p(x, C.c_float))
    return x[:n].copy()


def mlp_forward(mlp, x):
    nl, dims, Ws, bs, Wp, bp, sc = _mlp_args(mlp)
    x = _f32(x)
    y = np.empty(int(dims[-1]), dtype=np.float64)
    lib().orc_mlp_forward(C.c_int32(nl), _p(dims, C.c_int32), Wp, bp, _p(sc[0], C.c_float), _p(sc[1], C.c_float),
                          _p(sc[2], C.c_float), _p(sc[3], C.c_float), C.c_int32(mlp.get("act", 0)),
                          _p(x, C.c_float), _p(y, C.c_double))
    return y


def closure_mlp(mom, mlp, tau, min_count=2, relax_w=1.0, coef_old=None):
    mom = _f64(mom)
    ncell, stride = mom.shape
    assert stride in (13, 29)
    nl, dims, Ws, bs, Wp, bp, sc = _mlp_args(mlp)
    keep, tau_p, tau_s = _tau_args(tau, ncell)
    coef = np.empty((ncell, 9), dtype=np.float64)
    flags = np.zeros(ncell, dtype=np.uint32)
    old = _f64(coef_old) if coef_old is not None else np.zeros((ncell, 9))
    lib().orc_closure_mlp(C.c_int32(ncell), _p(mom, C.c_double), C.c_int32(stride), tau_p, C.c_double(tau_s),
                          C.c_int32(nl), _p(dims, C.c_int32), Wp, bp, _p(sc[0], C.c_float), _p(sc[1], C.c_float),
                          _p(sc[2], C.c_float), _p(sc[3], C.c_float), C.c_int32(mlp.get("act", 0)),
                          C.c_int32(mlp.get("feature_set", 0)), C.c_double(mlp.get("n_scale", 1.0)),
                          C.c_double(mlp.get("theta_ref", 0.5)), C.c_int32(min_count), C.c_double(relax_w),
                          _p(old, C.c_double), _p(coef, C.c_double), _p(flags, C.c_uint32))
    return coef, flags


# ---------------------------------------------------------------- S6
def philox4x32_10(ctr, key):
    ctr, key = _u32(ctr), _u32(key)
    out = np.empty(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(ctr, C.c_uint32), _p(key, C.c_uint32), _p(out, C.c_uint32))
    return out


def uniforms(pid, step, stream, seed):
    pid = _u32(np.atleast_1d(pid))
    out = np.empty((pid.shape[0], 4))
    u = (C.c_double * 4)()
    f = lib().orc_uniforms
    for i, p in enumerate(pid):
        f(C.c_uint32(int(p)), C.c_uint64(step), C.c_uint32(stream), C.c_uint64(seed), u)
        out[i] = u[:]
    return out


def normals(pid, step, stream, seed):
    pid = _u32(np.atleast_1d(pid))
    out = np.empty((pid.shape[0], 3))
    xi = (C.c_double * 3)()
    f = lib().orc_normals
    for i, p in enumerate(pid):
        f(C.c_uint32(int(p)), C.c_uint64(step), C.c_uint32(stream), C.c_uint64(seed), xi)
        out[i] = xi[:]
    return out


# ---------------------------------------------------------------- S5
def velocity_update(vx, vy, vz, pid, cell_start, mom, coef, tau, cfg, step, flags=None):
    """Returns new (vx, vy, vz) as fp32 copies and the flags array (OR-ed into ``flags`` if given)."""
    vx, vy, vz = _f32(vx).copy(), _f32(vy).copy(), _f32(vz).copy()
    pid, cell_start, mom = _u32(pid), _i32(cell_start), _f64(mom)
    coef = _f32(coef)
    ncell, stride = mom.shape
    keep, tau_p, tau_s = _tau_args(tau, ncell)
    fl = np.zeros(ncell, dtype=np.uint32) if flags is None else _u32(flags).copy()
    lib().orc_velocity_update(C.c_int32(ncell), _p(cell_start, C.c_int32), _p(vx, C.c_float), _p(vy, C.c_float),
                              _p(vz, C.c_float), _p(pid, C.c_uint32), _p(mom, C.c_double), C.c_int32(stride),
                              _p(coef, C.c_float), tau_p, C.c_double(tau_s), C.c_double(np.float32(cfg["dt"])),
                              C.c_double(np.float32(cfg["eps2_scale"])), C.c_int32(cfg["conserve_mode"]),
                              C.c_uint64(cfg["seed"]), C.c_uint64(step), _p(fl, C.c_uint32))
    return vx, vy, vz, fl


# ---------------------------------------------------------------- S7
def _wall_array(cfg):
    w = np.zeros((4, 5), dtype=np.float64)
    for k, row in enumerate(cfg["walls"]):
        w[k, 0] = row[0]
        w[k, 1:] = [np.float32(v) for v in row[1:]]
    return w


def stream_walls(state, cfg, step):
    out = {k: np.ascontiguousarray(state[k]).copy() for k in ("x", "y", "vx", "vy", "vz", "pid")}
    w = _wall_array(cfg)
    body = cfg.get("body")
    bk, bc = (1, body) if body else (0, (0.0, 0.0, 0.0, 0.0))
    lib().orc_stream_walls(C.c_int64(out["x"].shape[0]), _p(out["x"], C.c_float), _p(out["y"], C.c_float),
                           _p(out["vx"], C.c_float), _p(out["vy"], C.c_float), _p(out["vz"], C.c_float),
                           _p(out["pid"], C.c_uint32), C.c_int32(cfg["nx"]), C.c_int32(cfg["ny"]),
                           C.c_float(cfg["x0"]), C.c_float(cfg["y0"]), C.c_float(cfg["dx"]), C.c_float(cfg["dy"]),
                           C.c_float(cfg["dt"]), _p(w, C.c_double), C.c_int32(bk), C.c_float(bc[0]),
                           C.c_float(bc[1]), C.c_float(bc[2]), C.c_double(np.float32(bc[3])),
                           C.c_uint64(cfg["seed"]), C.c_uint64(step))
    return out


# ---------------------------------------------------------------- one step, Algorithm 1 / 2 order
def step(state, cfg, step_no, closure="exact", mlp=None, tau_cell=None, coef_old=None, relax_w=1.0):
    """stream -> walls -> sort -> moments -> closure -> update.
    tau_cell: None (cfg['tau']) or a callable N[ncell] -> tau[ncell] float32 (per-cell tau from the counts)."""
    s1 = stream_walls(state, cfg, step_no)
    s2, cell_start, perm = sort_by_cell(s1, cfg)
    full = closure == "exact"
    mom = cell_moments(s2["vx"], s2["vy"], s2["vz"], cell_start, 1 if full else 0)
    tau = np.float32(cfg["tau"]) if tau_cell is None else tau_cell(mom[:, 0])
    if full:
        coef, flags, _ = closure_exact(mom, tau, float(np.float32(cfg["eps2_scale"])), cfg["min_count"])
    else:
        coef, flags = closure_mlp(mom, mlp, tau, min_count=cfg.get("min_count_mlp", 2), relax_w=relax_w,
                                  coef_old=coef_old)
    coef32 = coef.astype(np.float32)
    vx, vy, vz, flags = velocity_update(s2["vx"], s2["vy"], s2["vz"], s2["pid"], cell_start, mom, coef32, tau, cfg,
                                        step_no, flags)
    s2["vx"], s2["vy"], s2["vz"] = vx, vy, vz
    return s2, dict(cell_start=cell_start, perm=perm, mom=mom, coef=coef32, flags=flags)
