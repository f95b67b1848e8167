"""Thin Python binding over the C-ABI library ``libfpcl.so`` (include/fpcl.h).  Argument marshalling only: every
step of the path runs in the library's CUDA kernels.  PyTorch supplies device memory and the current stream.

The module-level ``fp_*`` functions mirror the C entry points one to one (torch tensors in place of pointers);
``Context`` is a small convenience wrapper that allocates outputs.  There is no CPU fallback: if the library is
missing or a call fails, an exception is raised.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libfpcl.so")

FP_OK, FP_ERR_ARG, FP_ERR_STATE, FP_ERR_CUDA, FP_ERR_UNSUPPORTED = 0, -1, -2, -3, -4
FLAG_EMPTY, FLAG_LOWCOUNT, FLAG_SINGULAR, FLAG_ILLCOND, FLAG_ALPHA, FLAG_SKIPPED, FLAG_NONFINITE = 1, 2, 4, 8, 16, 32, 64

EXPORTS = ["fp_create", "fp_destroy", "fp_last_error", "fp_version", "fp_sort_by_cell", "fp_cell_moments",
           "fp_closure_exact", "fp_closure_mlp", "fp_velocity_update", "fp_stream_walls", "fp_step", "fp_step_host",
           "fp_timing_enable", "fp_timing_read", "fp_launch_count", "fp_set_mlp_tensor_cores", "fp_cell_diagnostics",
           "fp_average_results", "fp_cell_sixth_moment", "fp_reserve", "fp_check", "fp_set_slab", "fp_slab_partition",
           "fp_collide", "fp_set_reproducible", "fp_cell_moments_static", "fp_static_last_error"]
FP_STATIC_MAX_CELLS = 16384
NSTAGES = 6
STAGE_NAMES = ["stream_walls", "sort_keys", "gather", "moments", "closure", "update"]


class FpWall(C.Structure):
    _fields_ = [("kind", C.c_int32), ("theta_w", C.c_float), ("ux", C.c_float), ("uy", C.c_float), ("uz", C.c_float)]


class FpParams(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("x0", C.c_float), ("y0", C.c_float), ("dx", C.c_float),
                ("dy", C.c_float), ("max_particles", C.c_int64), ("dt", C.c_float), ("tau", C.c_float),
                ("eps2_scale", C.c_float), ("min_count", C.c_int32), ("min_count_mlp", C.c_int32),
                ("conserve_mode", C.c_int32), ("seed", C.c_uint64), ("wall", FpWall * 4), ("body_kind", C.c_int32),
                ("body_cx", C.c_float), ("body_cy", C.c_float), ("body_R", C.c_float), ("body_theta_w", C.c_float)]


class FpMlp(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("h_dims", C.POINTER(C.c_int32)), ("W", C.POINTER(C.c_void_p)),
                ("b", C.POINTER(C.c_void_p)), ("x_mean", C.c_void_p), ("x_scale", C.c_void_p),
                ("y_mean", C.c_void_p), ("y_scale", C.c_void_p), ("act", C.c_int32), ("feature_set", C.c_int32),
                ("n_scale", C.c_float), ("theta_ref", C.c_float)]


class FpclError(RuntimeError):
    pass


_lib = None


def load(path=None):
    """Load libfpcl.so (built by ``python -m paper_2606_15622_b200.build``).  Raises if it is missing."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or _LIBPATH
    if not os.path.exists(p):
        raise FpclError("libfpcl.so not found at %s: run `python -m paper_2606_15622_b200.build` "
                        "(there is no CPU fallback)" % p)
    lib = C.CDLL(p)
    vp, i64, i32, u64, f32 = C.c_void_p, C.c_int64, C.c_int32, C.c_uint64, C.c_float
    lib.fp_create.argtypes = [C.POINTER(vp), C.POINTER(FpParams)]
    lib.fp_destroy.argtypes = [vp]
    lib.fp_last_error.argtypes = [vp]
    lib.fp_last_error.restype = C.c_char_p
    lib.fp_version.restype = C.c_char_p
    lib.fp_sort_by_cell.argtypes = [vp, i64] + [vp] * 6 + [vp] * 6 + [vp, vp, vp]
    lib.fp_cell_moments.argtypes = [vp, i64, vp, vp, vp, vp, i32, vp, vp]
    lib.fp_closure_exact.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.fp_closure_mlp.argtypes = [vp, vp, i32, vp, C.POINTER(FpMlp), f32, vp, vp, vp]
    lib.fp_velocity_update.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, i32, vp, vp, u64, vp, vp]
    lib.fp_cell_diagnostics.argtypes = [vp, vp, C.c_double, C.c_double, C.c_double, vp, vp]
    lib.fp_average_results.argtypes = [vp, i64, vp, i64, vp, vp]
    lib.fp_cell_sixth_moment.argtypes = [vp, i64, vp, vp, vp, vp, vp, i32, vp, vp]
    lib.fp_stream_walls.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, u64, vp]
    lib.fp_step.argtypes = [vp, i64] + [vp] * 12 + [i32, C.POINTER(FpMlp), f32, i32, f32, vp, u64, vp, vp, vp, vp, vp]
    lib.fp_step_host.argtypes = [vp, i64] + [vp] * 6 + [i32, C.POINTER(FpMlp), f32, u64, vp, vp, vp, vp]
    lib.fp_timing_enable.argtypes = [vp, i32]
    lib.fp_timing_read.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(i32)]
    lib.fp_launch_count.argtypes = [vp]
    lib.fp_set_mlp_tensor_cores.argtypes = [vp, i32]
    lib.fp_reserve.argtypes = [vp, C.POINTER(FpMlp), i32]
    lib.fp_set_slab.argtypes = [vp, i32, i32]
    lib.fp_set_reproducible.argtypes = [vp, i32]
    lib.fp_slab_partition.argtypes = [vp, i64] + [vp] * 12 + [C.POINTER(i32), i32, vp, vp]
    lib.fp_collide.argtypes = [vp, i64] + [vp] * 12 + [i32, C.POINTER(FpMlp), f32, i32, f32, vp, u64, vp, vp, vp, vp, vp]
    lib.fp_check.argtypes = [vp, vp]
    for name in EXPORTS:
        if name not in ("fp_last_error", "fp_version", "fp_launch_count", "fp_static_last_error"):
            getattr(lib, name).restype = C.c_int
    lib.fp_launch_count.restype = C.c_uint64
    lib.fp_cell_moments_static.argtypes = [i64, vp, vp, vp, vp, i32, i32, vp, vp, vp]
    lib.fp_static_last_error.restype = C.c_char_p
    if path is None:
        _lib = lib
    return lib


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t, dtype=None, n=None):
    if t is None:
        return C.c_void_p(0)
    if not t.is_cuda or not t.is_contiguous():
        raise FpclError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise FpclError("expected dtype %s, got %s" % (dtype, t.dtype))
    if n is not None and t.numel() < n:
        raise FpclError("tensor too small: %d < %d" % (t.numel(), n))
    return C.c_void_p(t.data_ptr())


def _check(ctx, rc, what):
    if rc != 0:
        msg = load().fp_last_error(ctx).decode() if ctx else ""
        raise FpclError("%s failed with code %d: %s" % (what, rc, msg))


def params_from_config(cfg):
    """cfg: the plain dict of ``workloads.make_config``."""
    p = FpParams()
    p.nx, p.ny = cfg["nx"], cfg["ny"]
    p.x0, p.y0, p.dx, p.dy = cfg["x0"], cfg["y0"], cfg["dx"], cfg["dy"]
    p.max_particles = int(cfg["max_particles"])
    p.dt, p.tau, p.eps2_scale = cfg["dt"], cfg["tau"], cfg["eps2_scale"]
    p.min_count, p.min_count_mlp = cfg["min_count"], cfg.get("min_count_mlp", 2)
    p.conserve_mode, p.seed = cfg["conserve_mode"], cfg["seed"]
    for k, w in enumerate(cfg["walls"]):
        p.wall[k].kind, p.wall[k].theta_w, p.wall[k].ux, p.wall[k].uy, p.wall[k].uz = w
    body = cfg.get("body")
    if body:
        p.body_kind = 1
        p.body_cx, p.body_cy, p.body_R, p.body_theta_w = body
    return p


# ---------------------------------------------------------------------------------------------- C entry points
def fp_version():
    return load().fp_version().decode()


def fp_create(params):
    h = C.c_void_p()
    rc = load().fp_create(C.byref(h), C.byref(params))
    if rc != 0:
        raise FpclError("fp_create failed with code %d" % rc)
    return h


def fp_destroy(ctx):
    _check(None, load().fp_destroy(ctx), "fp_destroy")


def fp_sort_by_cell(ctx, np_, x, y, vx, vy, vz, pid, x_out, y_out, vx_out, vy_out, vz_out, pid_out, cell_start,
                    perm=None):
    f, u = torch.float32, torch.int32
    _check(ctx, load().fp_sort_by_cell(ctx, np_, _ptr(x, f, np_), _ptr(y, f, np_), _ptr(vx, f, np_), _ptr(vy, f, np_),
                                       _ptr(vz, f, np_), _ptr(pid, u, np_), _ptr(x_out, f, np_), _ptr(y_out, f, np_),
                                       _ptr(vx_out, f, np_), _ptr(vy_out, f, np_), _ptr(vz_out, f, np_),
                                       _ptr(pid_out, u, np_), _ptr(cell_start, u), _ptr(perm, u, np_), _stream()),
           "fp_sort_by_cell")


def fp_cell_moments(ctx, np_, vx, vy, vz, cell_start, mode, mom):
    f = torch.float32
    _check(ctx, load().fp_cell_moments(ctx, np_, _ptr(vx, f, np_), _ptr(vy, f, np_), _ptr(vz, f, np_),
                                       _ptr(cell_start, torch.int32), mode, _ptr(mom, torch.float64), _stream()),
           "fp_cell_moments")


def fp_cell_moments_static(np_, vx, vy, vz, cell_start, ncell, mode, mom, d_status=None):
    """The context-free, allocation-free moment gather (include/fpcl.h); marshalling only."""
    f = torch.float32
    lib = load()
    rc = lib.fp_cell_moments_static(np_, _ptr(vx, f, np_), _ptr(vy, f, np_), _ptr(vz, f, np_),
                                    _ptr(cell_start, torch.int32, ncell + 1), ncell, mode,
                                    _ptr(mom, torch.float64, ncell * (29 if mode else 13)), _ptr(d_status, torch.int32), _stream())
    if rc != 0:
        raise FpclError("fp_cell_moments_static failed with code %d: %s" % (rc, lib.fp_static_last_error().decode()))


def fp_closure_exact(ctx, mom_full, tau_cell, coef, flags, kappa_est=None):
    _check(ctx, load().fp_closure_exact(ctx, _ptr(mom_full, torch.float64), _ptr(tau_cell, torch.float32),
                                        _ptr(coef, torch.float32), _ptr(flags, torch.int32),
                                        _ptr(kappa_est, torch.float64), _stream()), "fp_closure_exact")


def fp_closure_mlp(ctx, mom, mom_stride, tau_cell, mlp, relax_w, coef, flags):
    _check(ctx, load().fp_closure_mlp(ctx, _ptr(mom, torch.float64), mom_stride, _ptr(tau_cell, torch.float32),
                                      C.byref(mlp.c_struct), relax_w, _ptr(coef, torch.float32),
                                      _ptr(flags, torch.int32), _stream()), "fp_closure_mlp")


def fp_velocity_update(ctx, np_, vx, vy, vz, pid, cell_start, mom, mom_stride, coef, tau_cell, step, flags):
    f = torch.float32
    _check(ctx, load().fp_velocity_update(ctx, np_, _ptr(vx, f, np_), _ptr(vy, f, np_), _ptr(vz, f, np_),
                                          _ptr(pid, torch.int32, np_), _ptr(cell_start, torch.int32),
                                          _ptr(mom, torch.float64), mom_stride, _ptr(coef, f), _ptr(tau_cell, f),
                                          step, _ptr(flags, torch.int32), _stream()), "fp_velocity_update")


def fp_cell_diagnostics(ctx, mom_full, theta_inf, n_inf, dg_inf, diag):
    _check(ctx, load().fp_cell_diagnostics(ctx, _ptr(mom_full, torch.float64), float(theta_inf), float(n_inf),
                                           float(dg_inf), _ptr(diag, torch.float64), _stream()), "fp_cell_diagnostics")


def fp_cell_sixth_moment(ctx, np_, vx, vy, vz, cell_start, mom, dm6):
    f = torch.float32
    _check(ctx, load().fp_cell_sixth_moment(ctx, np_, _ptr(vx, f, np_), _ptr(vy, f, np_), _ptr(vz, f, np_),
                                   _ptr(cell_start, torch.int32), _ptr(mom, torch.float64), mom.shape[1],
                                   _ptr(dm6, torch.float64), _stream()), "fp_cell_sixth_moment")


def fp_average_results(ctx, x, k, avg):
    _check(ctx, load().fp_average_results(ctx, x.numel(), _ptr(x, torch.float64), int(k),
                                          _ptr(avg, torch.float64, x.numel()), _stream()), "fp_average_results")


def fp_stream_walls(ctx, np_, x, y, vx, vy, vz, pid, step):
    f = torch.float32
    _check(ctx, load().fp_stream_walls(ctx, np_, _ptr(x, f, np_), _ptr(y, f, np_), _ptr(vx, f, np_), _ptr(vy, f, np_),
                                       _ptr(vz, f, np_), _ptr(pid, torch.int32, np_), step, _stream()),
           "fp_stream_walls")


def fp_step(ctx, np_, a, b, closure, mlp, relax_w, tau_mode, tau_ref_n, tau_cell, step, mom, coef, flags, cell_start):
    """a, b: dicts of x, y, vx, vy, vz (float32) and pid (int32 storage of the uint32 ids)."""
    f, u = torch.float32, torch.int32
    args = [_ptr(a[k], f, np_) for k in ("x", "y", "vx", "vy", "vz")] + [_ptr(a["pid"], u, np_)]
    args += [_ptr(b[k], f, np_) for k in ("x", "y", "vx", "vy", "vz")] + [_ptr(b["pid"], u, np_)]
    mp = C.byref(mlp.c_struct) if mlp is not None else C.POINTER(FpMlp)()
    _check(ctx, load().fp_step(ctx, np_, *args, closure, mp, relax_w, tau_mode, tau_ref_n, _ptr(tau_cell, f), step,
                               _ptr(mom, torch.float64), _ptr(coef, f), _ptr(flags, u), _ptr(cell_start, u),
                               _stream()), "fp_step")


def fp_collide(ctx, np_, a, b, closure, mlp, relax_w, tau_mode, tau_ref_n, tau_cell, step, mom, coef, flags, cell_start):
    """fp_step without the move: sort by cell -> moments -> closure -> update (positions of ``a`` are final)."""
    f, u = torch.float32, torch.int32
    args = [_ptr(a[k], f, np_) for k in ("x", "y", "vx", "vy", "vz")] + [_ptr(a["pid"], u, np_)]
    args += [_ptr(b[k], f, np_) for k in ("x", "y", "vx", "vy", "vz")] + [_ptr(b["pid"], u, np_)]
    mp = C.byref(mlp.c_struct) if mlp is not None else C.POINTER(FpMlp)()
    _check(ctx, load().fp_collide(ctx, np_, *args, closure, mp, relax_w, tau_mode, tau_ref_n, _ptr(tau_cell, f), step,
                                  _ptr(mom, torch.float64), _ptr(coef, f), _ptr(flags, u), _ptr(cell_start, u),
                                  _stream()), "fp_collide")


def fp_set_reproducible(ctx, on=True):
    _check(ctx, load().fp_set_reproducible(ctx, int(bool(on))), "fp_set_reproducible")


def fp_set_slab(ctx, row0, nrows):
    _check(ctx, load().fp_set_slab(ctx, int(row0), int(nrows)), "fp_set_slab")


def fp_slab_partition(ctx, np_, a, b, row_bounds, slab_start):
    """Stable partition of a's particles by destination slab into b; slab_start [nslabs+1] int32 on the device."""
    f, u = torch.float32, torch.int32
    args = [_ptr(a[k], f, np_) for k in ("x", "y", "vx", "vy", "vz")] + [_ptr(a["pid"], u, np_)]
    args += [_ptr(b[k], f, np_) for k in ("x", "y", "vx", "vy", "vz")] + [_ptr(b["pid"], u, np_)]
    rb = (C.c_int32 * len(row_bounds))(*[int(r) for r in row_bounds])
    _check(ctx, load().fp_slab_partition(ctx, np_, *args, rb, len(row_bounds) - 1, _ptr(slab_start, u), _stream()),
           "fp_slab_partition")


def _hptr(a, dtype):
    if a is None:
        return C.c_void_p(0)
    if isinstance(a, torch.Tensor):
        assert not a.is_cuda and a.is_contiguous()
        return C.c_void_p(a.data_ptr())
    assert a.dtype == dtype and a.flags["C_CONTIGUOUS"]
    return C.c_void_p(a.ctypes.data)


def fp_step_host(ctx, np_, h, closure, mlp, relax_w, step, h_coef=None, h_flags=None, h_cell_start=None):
    """h: dict of HOST arrays (numpy or CPU torch tensors, pinned or not) x, y, vx, vy, vz, pid; updated in place."""
    args = [_hptr(h[k], np.float32) for k in ("x", "y", "vx", "vy", "vz")] + [_hptr(h["pid"], np.uint32)]
    mp = C.byref(mlp.c_struct) if mlp is not None else C.POINTER(FpMlp)()
    _check(ctx, load().fp_step_host(ctx, np_, *args, closure, mp, relax_w, step, _hptr(h_coef, np.float32),
                                    _hptr(h_flags, np.uint32), _hptr(h_cell_start, np.int32), _stream()),
           "fp_step_host")


def fp_timing_enable(ctx, max_steps):
    _check(ctx, load().fp_timing_enable(ctx, max_steps), "fp_timing_enable")


def fp_timing_read(ctx, max_steps):
    """Returns an array [nsteps, NSTAGES] of stage durations in ms (see STAGE_NAMES)."""
    buf = (C.c_float * (max_steps * NSTAGES))()
    n = C.c_int32(0)
    _check(ctx, load().fp_timing_read(ctx, buf, C.byref(n)), "fp_timing_read")
    return np.frombuffer(buf, dtype=np.float32)[: n.value * NSTAGES].reshape(n.value, NSTAGES).copy()


def fp_set_mlp_tensor_cores(ctx, enable):
    _check(ctx, load().fp_set_mlp_tensor_cores(ctx, int(enable)), "fp_set_mlp_tensor_cores")


def fp_launch_count(ctx):
    return int(load().fp_launch_count(ctx))


def fp_reserve(ctx, mlp=None, host_staging=False):
    _check(ctx, load().fp_reserve(ctx, C.byref(mlp.c_struct) if mlp is not None else None, int(bool(host_staging))),
           "fp_reserve")


def fp_check(ctx):
    _check(ctx, load().fp_check(ctx, _stream()), "fp_check")


# ---------------------------------------------------------------------------------------------- conveniences
class Mlp:
    """Device copy of an MLP parameter dict (``workloads.xavier_mlp`` layout) plus its ``fp_mlp`` struct."""

    def __init__(self, mlp, device="cuda"):
        dims = [int(d) for d in mlp["dims"]]
        self.dims = dims
        nl = len(dims) - 1
        self.W = [torch.as_tensor(np.ascontiguousarray(w, dtype=np.float32)).to(device) for w in mlp["W"]]
        self.b = [torch.as_tensor(np.ascontiguousarray(b, dtype=np.float32)).to(device) for b in mlp["b"]]
        self.scalers = [torch.as_tensor(np.ascontiguousarray(mlp[k], dtype=np.float32)).to(device)
                        for k in ("x_mean", "x_scale", "y_mean", "y_scale")]
        self._dims = (C.c_int32 * (nl + 1))(*dims)
        self._W = (C.c_void_p * nl)(*[w.data_ptr() for w in self.W])
        self._b = (C.c_void_p * nl)(*[b.data_ptr() for b in self.b])
        s = FpMlp()
        s.n_layers = nl
        s.h_dims = C.cast(self._dims, C.POINTER(C.c_int32))
        s.W = C.cast(self._W, C.POINTER(C.c_void_p))
        s.b = C.cast(self._b, C.POINTER(C.c_void_p))
        s.x_mean, s.x_scale, s.y_mean, s.y_scale = [t.data_ptr() for t in self.scalers]
        s.act, s.feature_set = int(mlp.get("act", 0)), int(mlp.get("feature_set", 0))
        s.n_scale, s.theta_ref = float(mlp.get("n_scale", 1.0)), float(mlp.get("theta_ref", 0.5))
        self.c_struct = s


def to_device(state, device="cuda"):
    """numpy state dict (x, y, vx, vy, vz float32; pid uint32) -> dict of CUDA tensors (pid stored as int32 bits)."""
    out = {k: torch.from_numpy(np.ascontiguousarray(state[k], dtype=np.float32)).to(device)
           for k in ("x", "y", "vx", "vy", "vz")}
    out["pid"] = torch.from_numpy(np.ascontiguousarray(state["pid"], dtype=np.uint32).view(np.int32)).to(device)
    return out


def to_host(state):
    out = {k: state[k].cpu().numpy() for k in ("x", "y", "vx", "vy", "vz")}
    out["pid"] = state["pid"].cpu().numpy().view(np.uint32)
    return out


class Context:
    """Owns an ``fp_ctx`` and allocates outputs; each method is one C call."""

    def __init__(self, cfg, device="cuda"):
        if not torch.cuda.is_available():
            raise FpclError("fpcl needs a CUDA device (there is no CPU fallback)")
        self.cfg = dict(cfg)
        self.device = torch.device(device)
        self.ncell = int(cfg["nx"]) * int(cfg["ny"])
        self.params = params_from_config(cfg)
        with torch.cuda.device(self.device):
            self.h = fp_create(self.params)

    def close(self):
        if self.h is not None:
            fp_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _empty_like_state(self, n):
        out = {k: torch.empty(n, dtype=torch.float32, device=self.device) for k in ("x", "y", "vx", "vy", "vz")}
        out["pid"] = torch.empty(n, dtype=torch.int32, device=self.device)
        return out

    def sort_by_cell(self, s, want_perm=True):
        n = s["x"].numel()
        o = self._empty_like_state(n)
        cell_start = torch.empty(self.ncell + 1, dtype=torch.int32, device=self.device)
        perm = torch.empty(n, dtype=torch.int32, device=self.device) if want_perm else None
        fp_sort_by_cell(self.h, n, s["x"], s["y"], s["vx"], s["vy"], s["vz"], s["pid"], o["x"], o["y"], o["vx"],
                        o["vy"], o["vz"], o["pid"], cell_start, perm)
        return o, cell_start, perm

    def cell_moments(self, vx, vy, vz, cell_start, mode, out=None):
        mom = out if out is not None else torch.empty((self.ncell, 29 if mode else 13), dtype=torch.float64,
                                                      device=self.device)
        fp_cell_moments(self.h, vx.numel(), vx, vy, vz, cell_start, mode, mom)
        return mom

    def closure_exact(self, mom, tau_cell=None, want_kappa=False):
        coef = torch.empty((self.ncell, 9), dtype=torch.float32, device=self.device)
        flags = torch.empty(self.ncell, dtype=torch.int32, device=self.device)
        kap = torch.empty(self.ncell, dtype=torch.float64, device=self.device) if want_kappa else None
        fp_closure_exact(self.h, mom, tau_cell, coef, flags, kap)
        return (coef, flags, kap) if want_kappa else (coef, flags)

    def closure_mlp(self, mom, mlp, tau_cell=None, relax_w=1.0, coef=None):
        if coef is None:
            coef = torch.zeros((self.ncell, 9), dtype=torch.float32, device=self.device)
        flags = torch.empty(self.ncell, dtype=torch.int32, device=self.device)
        fp_closure_mlp(self.h, mom, mom.shape[1], tau_cell, mlp, relax_w, coef, flags)
        return coef, flags

    def cell_diagnostics(self, mom_full, theta_inf=0.5, n_inf=1.0, dg_inf=0.0, out=None):
        diag = out if out is not None else torch.empty((self.ncell, 16), dtype=torch.float64, device=self.device)
        fp_cell_diagnostics(self.h, mom_full, theta_inf, n_inf, dg_inf, diag)
        return diag

    def velocity_update(self, vx, vy, vz, pid, cell_start, mom, coef, step, flags, tau_cell=None):
        fp_velocity_update(self.h, vx.numel(), vx, vy, vz, pid, cell_start, mom, mom.shape[1], coef, tau_cell, step,
                           flags)

    def stream_walls(self, s, step):
        fp_stream_walls(self.h, s["x"].numel(), s["x"], s["y"], s["vx"], s["vy"], s["vz"], s["pid"], step)

    def alloc_step_outputs(self, closure):
        return dict(mom=torch.empty((self.ncell, 29 if closure == 0 else 13), dtype=torch.float64, device=self.device),
                    coef=torch.zeros((self.ncell, 9), dtype=torch.float32, device=self.device),
                    flags=torch.zeros(self.ncell, dtype=torch.int32, device=self.device),
                    cell_start=torch.empty(self.ncell + 1, dtype=torch.int32, device=self.device))

    def step(self, a, b, step, out, closure=0, mlp=None, relax_w=1.0, tau_mode=0, tau_ref_n=0.0, tau_cell=None):
        fp_step(self.h, a["x"].numel(), a, b, closure, mlp, relax_w, tau_mode, tau_ref_n, tau_cell, step, out["mom"],
                out["coef"], out["flags"], out["cell_start"])

    def step_host(self, h, step, closure=0, mlp=None, relax_w=1.0, h_coef=None, h_flags=None, h_cell_start=None):
        fp_step_host(self.h, h["x"].shape[0], h, closure, mlp, relax_w, step, h_coef, h_flags, h_cell_start)
