"""GPU-vs-oracle parity for the particle stages (a0/a1 stream+walls, a6 update), the composed fp_step (a7), the
host-buffer entry point, and a full-size check at BASELINE config 3 (4M particles) in the launch configuration
bench.py times."""
import numpy as np
import pytest

from parity_util import abs_moments, coef_ratio, moment_ratio, velocity_ratio

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_15622_b200 import fpcl
    fpcl.load()
    return fpcl


@pytest.fixture(scope="module")
def wl():
    from paper_2606_15622_b200 import workloads
    return workloads


def _theta(mom):
    return (mom[:, 4] + mom[:, 7] + mom[:, 9]) / 3.0


def _bits(a):
    return np.ascontiguousarray(a).view(np.uint32)


# ------------------------------------------------------------------------------------------------ a6 update
@pytest.mark.parametrize("case", ["couette-exact", "ragged-exact", "ragged-mlp", "ragged1d-exact", "highppc-exact", "highppc-mlp"])
@pytest.mark.parametrize("mode", [0, 1])
def test_velocity_update(gpu, wl, orc, case, mode):
    import torch
    name, closure = case.split("-")
    cfg, st = {"couette": wl.couette, "ragged": wl.ragged,
               "ragged1d": lambda: wl.ragged(nx=64, ny=1, seed=11, mean_ppc=150.0),
               # few, huge cells (ragged: empty and 1-3 particle cells, cells of up to ~12,000): update_seg.cuh
               "highppc": lambda: wl.ragged(nx=9, ny=7, seed=31, mean_ppc=900.0)}[name]()
    cfg = dict(cfg, conserve_mode=mode)
    s, cs, _ = orc.sort_by_cell(st, cfg)
    ncell = cs.shape[0] - 1
    rng = np.random.default_rng(17)
    tau = rng.uniform(0.3, 2.0, size=ncell).astype(np.float32) if name in ("ragged", "highppc") else cfg["tau"]
    if closure == "exact":
        mom = orc.cell_moments(s["vx"], s["vy"], s["vz"], cs, 1)
        coef, flags, _ = orc.closure_exact(mom, tau, cfg["eps2_scale"], cfg["min_count"])
    else:
        mom = orc.cell_moments(s["vx"], s["vy"], s["vz"], cs, 0)
        mlp = wl.xavier_mlp(n_scale=1.0 / 40.0, tau=cfg["tau"], bias_scale=0.1)
        coef, flags = orc.closure_mlp(mom, mlp, tau, min_count=2)
    coef32 = coef.astype(np.float32)
    step = (1 << 33) + 12345
    rvx, rvy, rvz, rfl = orc.velocity_update(s["vx"], s["vy"], s["vz"], s["pid"], cs, mom, coef32, tau, cfg, step, flags)
    ctx = gpu.Context(cfg)
    d = gpu.to_device(s)
    fl = torch.from_numpy(flags.view(np.int32).copy()).cuda()
    tau_d = None if np.ndim(tau) == 0 else torch.from_numpy(tau).cuda()
    ctx.velocity_update(d["vx"], d["vy"], d["vz"], d["pid"], torch.from_numpy(cs).cuda(), torch.from_numpy(mom).cuda(),
                        torch.from_numpy(coef32).cuda(), step, fl, tau_cell=tau_d)
    got = (d["vx"].cpu().numpy(), d["vy"].cpu().numpy(), d["vz"].cpu().numpy())
    assert np.array_equal(fl.cpu().numpy().view(np.uint32), rfl)
    r = velocity_ratio(got, (rvx, rvy, rvz), cs, _theta(mom))
    print("update %s mode %d: worst err/allowed %.3f" % (case, mode, r))
    assert r <= 1.0
    if mode == 1:   # per-cell momentum and energy of the fp32 outputs, evaluated in fp64
        n = np.diff(cs)
        act = (n >= 2) & (_theta(mom) > 0)
        seg = np.repeat(np.arange(ncell), n)
        for comp, (g, o) in enumerate(zip(got, (s["vx"], s["vy"], s["vz"]))):
            pg = np.bincount(seg, weights=g.astype(np.float64), minlength=ncell)
            po = np.bincount(seg, weights=o.astype(np.float64), minlength=ncell)
            scale = np.sqrt(np.maximum(_theta(mom), 1e-300)) * np.maximum(n, 1)
            assert (np.abs(pg - po)[act] / scale[act]).max() < 2e-6
        eg = sum(np.bincount(seg, weights=g.astype(np.float64) ** 2, minlength=ncell) for g in got)
        eo = sum(np.bincount(seg, weights=o.astype(np.float64) ** 2, minlength=ncell) for o in (s["vx"], s["vy"], s["vz"]))
        assert (np.abs(eg - eo)[act] / eo[act]).max() < 2e-6
    ctx.close()


# ------------------------------------------------------------------------------------------------ a0 + a1
def _cyl_small(wl):
    cfg, st, tau_cell = wl.cylinder(nx=80, ny=60, seed=5, target=200_000)
    return cfg, st, tau_cell


@pytest.mark.parametrize("name", ["couette", "cavity", "periodic", "cylinder", "reservoir_subsonic"])
def test_stream_walls(gpu, wl, orc, name):
    if name == "couette":
        cfg, st = wl.couette()
        cfg = dict(cfg, dt=np.float32(0.05))
    elif name == "cavity":
        cfg, st = wl.cavity(n=24, ppc=40, seed=5)
        cfg = dict(cfg, dt=float(np.float32(0.03)))          # long step: many wall and corner hits
    elif name == "periodic":
        w = [(wl.WALL_PERIODIC, 0.5, 0, 0, 0)] * 2 + [(wl.WALL_DIFFUSE, 0.7, 0.1, 0, 0.2), (wl.WALL_NONE, 0.5, 0, 0, 0)]
        cfg, st = wl.ragged(nx=20, ny=10, seed=2, mean_ppc=30.0, walls=w)
        cfg = dict(cfg, dt=float(np.float32(0.05)))
    elif name == "reservoir_subsonic":
        # freestream faces at U_inf = 0.25 sqrt(theta)-ish: the acceptance-rejection of the re-insertion rejects often, so
        # the accept / reject decisions of the two sides (fp32 kernel, fp64 oracle) are compared on thousands of draws
        w = [(wl.WALL_INFLOW, 0.5, 0.25, -0.2, 0.1)] * 4
        cfg, st = wl.ragged(nx=20, ny=10, seed=4, mean_ppc=60.0, walls=w)
        cfg = dict(cfg, dt=float(np.float32(0.08)))
    else:
        cfg, st, _ = _cyl_small(wl)                      # Mach-10 freestream faces + the body
        cfg = dict(cfg, dt=float(np.float32(0.4)))
    cfg = dict(cfg, dt=float(np.float32(cfg["dt"])))
    step = 7
    ref = orc.stream_walls(st, cfg, step)
    ctx = gpu.Context(cfg)
    d = gpu.to_device(st)
    ctx.stream_walls(d, step)
    got = gpu.to_host(d)
    assert np.array_equal(_bits(got["x"]), _bits(ref["x"]))
    assert np.array_equal(_bits(got["y"]), _bits(ref["y"]))
    hit = (_bits(ref["vx"]) != _bits(st["vx"])) | (_bits(ref["vy"]) != _bits(st["vy"])) | (_bits(ref["vz"]) != _bits(st["vz"]))
    print("stream_walls %s: %d of %d particles re-emitted" % (name, int(hit.sum()), hit.size))
    assert hit.sum() > 0 or name == "none"
    for k in ("vx", "vy", "vz"):
        assert np.array_equal(_bits(got[k])[~hit], _bits(st[k])[~hit])           # untouched particles keep their bits
        tw = max(w[1] for w in cfg["walls"]) if cfg.get("body") is None else max(cfg["body"][3], 0.5)
        allowed = 1e-6 * np.maximum(np.abs(ref[k][hit].astype(np.float64)), np.sqrt(tw))
        assert (np.abs(got[k][hit].astype(np.float64) - ref[k][hit]) <= allowed).all(), k
    ctx.close()


def test_stream_walls_unaligned(gpu, wl, orc):
    """Array views that start 4 bytes past a 16-byte boundary and a particle count that is not a multiple of 4
    (nor of the warp size) must give the same bits as aligned arrays."""
    import torch
    cfg, st = wl.cavity(n=16, ppc=37, seed=9)
    cfg = dict(cfg, dt=float(np.float32(0.03)))
    keep = st["x"].shape[0] - 3                     # 9469 particles: not a multiple of 4
    st = {k: v[:keep].copy() for k, v in st.items()}
    ref = orc.stream_walls(st, cfg, 5)
    ctx = gpu.Context(cfg)
    for off in (0, 1):
        d = {}
        for k, v in st.items():
            buf = torch.empty(keep + 4, dtype=torch.int32 if k == "pid" else torch.float32, device="cuda")
            d[k] = buf[off:off + keep]
            d[k].copy_(torch.from_numpy(v.view(np.int32) if k == "pid" else v))
        ctx.stream_walls(d, 5)
        got = {k: v.cpu().numpy() for k, v in d.items()}
        assert np.array_equal(_bits(got["x"]), _bits(ref["x"])), off
        assert np.array_equal(_bits(got["y"]), _bits(ref["y"])), off
        hit = (_bits(ref["vx"]) != _bits(st["vx"])) | (_bits(ref["vy"]) != _bits(st["vy"])) | (_bits(ref["vz"]) != _bits(st["vz"]))
        assert hit.sum() > 0
        for k in ("vx", "vy", "vz"):
            assert np.array_equal(_bits(got[k])[~hit], _bits(st[k])[~hit])
            allowed = 1e-6 * np.maximum(np.abs(ref[k][hit].astype(np.float64)), np.sqrt(0.5))
            assert (np.abs(got[k][hit].astype(np.float64) - ref[k][hit]) <= allowed).all(), (off, k)
    ctx.close()


# ------------------------------------------------------------------------------------------------ a7 fp_step
def _one_step(gpu, orc, cfg, st, closure, mlp, step_no, tau_fn=None, tau_ref_n=0.0):
    import torch
    ctx = gpu.Context(cfg)
    a = gpu.to_device(st)
    b = {k: torch.empty_like(v) for k, v in a.items()}
    out = ctx.alloc_step_outputs(closure)
    dm = gpu.Mlp(mlp) if mlp is not None else None
    tau_cell = torch.empty(ctx.ncell, dtype=torch.float32, device="cuda") if tau_fn is not None else None
    ctx.step(a, b, step_no, out, closure=closure, mlp=dm, tau_mode=1 if tau_fn is not None else 0,
             tau_ref_n=tau_ref_n, tau_cell=tau_cell)
    torch.cuda.synchronize()
    got = gpu.to_host(b)
    res = {k: v.cpu().numpy() for k, v in out.items()}
    ctx.close()
    ref, aux = orc.step(st, cfg, step_no, closure="exact" if closure == 0 else "mlp", mlp=mlp, tau_cell=tau_fn)
    return got, res, ref, aux


@pytest.mark.parametrize("name", ["couette", "cavity", "cylinder"])
@pytest.mark.parametrize("closure", [0, 1, 2])
def test_step_one(gpu, wl, orc, name, closure):
    # closure 2 = the surrogate step with the paper's own 16-256x4-9 network (tcgen05 kernel inside fp_step)
    wide = closure == 2
    if wide and name != "cavity":
        pytest.skip("wide surrogate: cavity only")
    closure = min(closure, 1)
    tau_fn, tau_ref_n = None, 0.0
    if name == "couette":
        cfg, st = wl.couette()
    elif name == "cavity":
        cfg, st = wl.cavity(n=32, ppc=60, seed=3)
    else:
        cfg, st, _ = _cyl_small(wl)
        tau_ref_n = float(np.float32(cfg["tau"] * cfg["ppc_inf"]))
        tau_default = np.float32(cfg["tau"])

        def tau_fn(N):
            with np.errstate(divide="ignore"):
                return np.where(N > 0, np.float32(tau_ref_n) / np.maximum(N, 1).astype(np.float32), tau_default).astype(np.float32)
    mlp = wl.xavier_mlp(n_scale=1.0 / 100.0, tau=cfg["tau"], bias_scale=0.1) if closure == 1 else None
    if wide:
        mlp = wl.xavier_mlp(dims=(16, 256, 256, 256, 256, 9), act=1, feature_set=1, n_scale=1.0 / 100.0, tau=cfg["tau"],
                            bias_scale=0.1)
    got, res, ref, aux = _one_step(gpu, orc, cfg, st, closure, mlp, 3, tau_fn, tau_ref_n)
    # integer outputs: bit-exact
    assert np.array_equal(res["cell_start"], aux["cell_start"])
    assert np.array_equal(got["pid"], ref["pid"])
    assert np.array_equal(_bits(got["x"]), _bits(ref["x"])) and np.array_equal(_bits(got["y"]), _bits(ref["y"]))
    # moments: 1e-6 where both sides saw bit-identical velocities; cells holding a re-emitted particle (whose fp32
    # wall draw may differ from the oracle's fp64 one by up to 1e-6, R7) are compared at 1e-5
    mid = orc.stream_walls(st, cfg, 3)
    hit = (_bits(mid["vx"]) != _bits(st["vx"])) | (_bits(mid["vy"]) != _bits(st["vy"])) | (_bits(mid["vz"]) != _bits(st["vz"]))
    touched = np.zeros(aux["mom"].shape[0], dtype=bool)
    touched[orc.cell_index(mid["x"][hit], mid["y"][hit], cfg)] = True
    pre, pre_cs, _ = orc.sort_by_cell(mid, cfg)               # the oracle's sorted pre-update particles
    am = abs_moments(pre["vx"], pre["vy"], pre["vz"], pre_cs, aux["mom"])
    rm0 = moment_ratio(res["mom"], aux["mom"], 1e-6, absmom=am, mask=~touched)
    rm1 = moment_ratio(res["mom"], aux["mom"], 1e-5, absmom=am, mask=touched)
    rm = max(rm0, rm1)
    delta_mom = np.where(touched, rm1 * 1e-5, rm0 * 1e-6)      # measured relative mismatch of the two sides' moments
    assert rm <= 1.0
    theta = _theta(aux["mom"])
    tau = cfg["tau"] if tau_fn is None else tau_fn(aux["mom"][:, 0])
    hard = orc.FLAG_EMPTY | orc.FLAG_LOWCOUNT | orc.FLAG_SINGULAR | orc.FLAG_SKIPPED
    gflags = res["flags"].view(np.uint32)
    assert np.array_equal(gflags & hard, aux["flags"] & hard)
    if closure == 0:
        # the two closures start from moments that differ by delta_mom (measured above, ~1e-7): per cell the coefficient
        # tolerance is max(1e-5, 30 kappa delta_mom) on every cell below the kappa < 1e8 line.  (SURVEY 8(c) S3-d wrote
        # 10 kappa delta_mom; the perturbation bound is |dy|/|y| <= kappa (|dA|/|A| + |db|/|b|) = 2 kappa delta in one
        # norm, and delta_mom is measured per entry against its own scale while kappa_1 is a 1-norm quantity of a 9x9
        # system: up to another factor 9.  Measured: 11 kappa delta_mom on the cavity, hence 30.)
        _, _, kappa = orc.closure_exact(aux["mom"], tau, cfg["eps2_scale"], cfg["min_count"])
        good = ((aux["flags"] & (hard | orc.FLAG_ILLCOND)) == 0) & (kappa < 1e8)
        rc = coef_ratio(res["coef"], aux["coef"], tau, theta, np.maximum(1e-5, 30.0 * kappa * delta_mom), mask=good)
        # Mach-10 shock-band cells have an O(1) cubic term eps2 c^3 tau: the ~1e-7 mismatch of the two sides' moments
        # (U, theta, h, eps2) is amplified ~100x on its way to the velocities (the stage test feeds identical moments)
        tolv = 1e-4 if name == "cylinder" else 2e-5
    else:
        good = (aux["flags"] & orc.FLAG_EMPTY) == 0
        # benchmark-shape surrogate runs on the tensor cores (3xTF32, ~1e-5 of the output scale; see test_closure_mlp)
        rc = coef_ratio(res["coef"], aux["coef"], tau, theta, 1e-4 if wide else 3e-5, mask=good)
        # the surrogate standardises its inputs by 0.05-0.3, so at Mach 10 (|U| = 9) the ~1e-7 relative mismatch
        # of the two sides' moments reaches the coefficients at ~1e-5 and the velocities through (1 - E1) tau N
        tolv = 5e-5 if name == "cylinder" else (1.5e-5 if wide else 4e-6)
    n = np.diff(aux["cell_start"])
    pm = np.repeat(good, n)
    cs_good = np.concatenate([[0], np.cumsum(n[good])]).astype(np.int64)
    rv = velocity_ratio(tuple(got[k][pm] for k in ("vx", "vy", "vz")), tuple(ref[k][pm] for k in ("vx", "vy", "vz")),
                        cs_good, theta[good], tolv)
    print("step %s closure %d: moments %.3f coef %.3g velocities %.3f (of tol %.0e) over %d/%d cells"
          % (name, closure, rm, rc, rv, tolv, int(good.sum()), good.size))
    assert rc <= 1.0 and rv <= 1.0
    for k in ("vx", "vy", "vz"):
        assert np.isfinite(got[k]).all()


def test_step_host(gpu, wl, orc):
    """fp_step_host: host buffers in, host buffers out, same result as the device-resident call."""
    import torch
    cfg, st = wl.cavity(n=16, ppc=50, seed=9)
    ctx = gpu.Context(cfg)
    a = gpu.to_device(st)
    b = {k: torch.empty_like(v) for k, v in a.items()}
    out = ctx.alloc_step_outputs(0)
    ctx.step(a, b, 5, out, closure=0)
    want = gpu.to_host(b)
    h = {k: np.ascontiguousarray(v).copy() for k, v in st.items()}
    ncell = ctx.ncell
    hc, hf, hs = np.empty((ncell, 9), np.float32), np.empty(ncell, np.uint32), np.empty(ncell + 1, np.int32)
    ctx.step_host(h, 5, closure=0, h_coef=hc, h_flags=hf, h_cell_start=hs)
    for k in ("x", "y", "vx", "vy", "vz", "pid"):
        assert np.array_equal(_bits(h[k]), _bits(want[k])), k
    assert np.array_equal(hs, out["cell_start"].cpu().numpy())
    assert np.array_equal(hc, out["coef"].cpu().numpy())
    ctx.close()


def test_step_host_pinned_large_with_walls(gpu, wl):
    """fp_step_host with PINNED host buffers and 1M particles at a large time step (many wall re-emissions, which
    rewrite vx, vy, vz in the stream kernel): bit-identical to the device-resident fp_step.  Guards the ordering of the
    uploads against the first kernel (a vz copy still in flight used to be able to overwrite the re-drawn vz)."""
    import torch
    cfg, st = wl.cavity(n=100, ppc=100, seed=12)
    cfg["dt"] = float(np.float32(0.02))                                  # ~2 cells per step: a few percent hit a wall
    ctx = gpu.Context(cfg)
    gpu.fp_reserve(ctx.h, None, True)                                    # staging buffers up front
    a = gpu.to_device(st)
    b = {k: torch.empty_like(v) for k, v in a.items()}
    out = ctx.alloc_step_outputs(0)
    ctx.step(a, b, 3, out, closure=0)
    want = gpu.to_host(b)
    moved = (np.abs(st["vz"][want["pid"]] - want["vz"]) > 0).mean()
    h = {k: torch.from_numpy(np.ascontiguousarray(v).copy()).pin_memory() for k, v in st.items() if k != "pid"}
    h["pid"] = torch.from_numpy(st["pid"].view(np.int32).copy()).pin_memory()
    for rep in range(3):                                                 # a race would not show every time
        for k, v in st.items():
            h[k].copy_(torch.from_numpy(v.view(np.int32) if k == "pid" else v))
        hn = {k: (v.numpy().view(np.uint32) if k == "pid" else v.numpy()) for k, v in h.items()}
        ctx.step_host(hn, 3, closure=0)
        for k in ("x", "y", "vx", "vy", "vz", "pid"):
            assert np.array_equal(_bits(hn[k]), _bits(want[k])), (k, rep)
    assert moved > 0.9                                                   # the update touched the velocities at all
    ctx.close()


def test_unsorted_cell_start_is_a_state_error(gpu, wl):
    """cell_start that is not a monotone prefix ending at np: the cells concerned are skipped on the device, the sticky
    state word makes the NEXT entry point return FP_ERR_STATE, fp_check reports and clears it (include/fpcl.h)."""
    import torch
    cfg, st = wl.cavity(n=12, ppc=40, seed=4)
    ctx = gpu.Context(cfg)
    a = gpu.to_device(st)
    b = {k: torch.empty_like(v) for k, v in a.items()}
    out = ctx.alloc_step_outputs(0)
    ctx.step(a, b, 0, out, closure=0)
    cs = out["cell_start"].clone()
    good = ctx.cell_moments(b["vx"], b["vy"], b["vz"], cs, 1)
    gpu.fp_check(ctx.h)                                                  # clean so far
    for kind in ("swap", "end", "negative"):
        bad = cs.clone()
        if kind == "swap":
            bad[40], bad[41] = cs[41] + 7, cs[40]
        elif kind == "end":
            bad[-1] = cs[-1] - 1
        else:
            bad[5] = -3
        mom = ctx.cell_moments(b["vx"], b["vy"], b["vz"], bad, 1)        # asynchronous: returns FP_OK
        torch.cuda.synchronize()
        assert torch.isfinite(mom).all()
        with pytest.raises(gpu.FpclError, match="code -2"):
            ctx.cell_moments(b["vx"], b["vy"], b["vz"], cs, 1)
        with pytest.raises(gpu.FpclError, match="code -2"):
            gpu.fp_check(ctx.h)
        gpu.fp_check(ctx.h)                                              # cleared
        v = [b[k].clone() for k in ("vx", "vy", "vz")]
        fl = out["flags"].clone()
        ctx.velocity_update(v[0], v[1], v[2], b["pid"], bad, good, out["coef"], 9, fl)
        torch.cuda.synchronize()
        assert all(torch.isfinite(x).all() for x in v)
        with pytest.raises(gpu.FpclError, match="code -2"):
            gpu.fp_check(ctx.h)
    again = ctx.cell_moments(b["vx"], b["vy"], b["vz"], cs, 1)
    assert torch.equal(again, good)
    ctx.close()


def test_multi_step_statistics(gpu, wl, orc):
    """100 Couette steps (BASELINE config 1) with each closure: particle count and ids conserved, no non-finite value,
    temperature stays put, and the mean profile agrees with the oracle's own 100-step run statistically."""
    import torch
    cfg, st = wl.couette()
    nsteps = 100
    for closure in (0, 1):
        mlp = wl.xavier_mlp(n_scale=0.01, tau=cfg["tau"]) if closure == 1 else None
        ctx = gpu.Context(cfg)
        a = gpu.to_device(st)
        b = {k: torch.empty_like(v) for k, v in a.items()}
        out = ctx.alloc_step_outputs(closure)
        dm = gpu.Mlp(mlp) if mlp is not None else None
        for it in range(nsteps):
            ctx.step(a, b, it, out, closure=closure, mlp=dm)
            a, b = b, a
        g = gpu.to_host(a)
        s = {k: v.copy() for k, v in st.items()}
        for it in range(nsteps):
            s, _ = orc.step(s, cfg, it, closure="exact" if closure == 0 else "mlp", mlp=mlp)
        assert np.array_equal(np.sort(g["pid"]), np.arange(st["pid"].shape[0], dtype=np.uint32))
        for k in ("x", "vx", "vy", "vz"):
            assert np.isfinite(g[k]).all()
        assert (g["x"] >= 0).all() and (g["x"] < 1).all()
        Tg = (g["vx"].astype(np.float64) ** 2 + (g["vy"].astype(np.float64)) ** 2 + g["vz"].astype(np.float64) ** 2).mean() / 3
        To = (s["vx"].astype(np.float64) ** 2 + (s["vy"].astype(np.float64)) ** 2 + s["vz"].astype(np.float64) ** 2).mean() / 3
        print("couette 100 steps closure %d: <v^2>/3 gpu %.4f oracle %.4f" % (closure, Tg, To))
        assert abs(Tg - To) < 0.03
        # shear profile: slope of <v_y>(x) agrees within statistical noise (5000 particles: sigma ~ 0.035 on the slope)
        sg = np.polyfit(g["x"].astype(np.float64), g["vy"].astype(np.float64), 1)[0]
        so = np.polyfit(s["x"].astype(np.float64), s["vy"].astype(np.float64), 1)[0]
        assert abs(sg - so) < 0.2
        ctx.close()


# ------------------------------------------------------------------------------------------------ full size
@pytest.mark.parametrize("case", ["c3_4m", "c4_8m", "c5_20m"])
def test_full_size(gpu, wl, orc, case):
    """BASELINE configs at their full sizes, every stage against the oracle on the full arrays, in the launch
    configuration bench.py times: C3 (200x200 cells x 100 ppc = 4M particles), C4 at 200 ppc (8M particles: the packed
    sort with 23 index bits, G = 16 lanes per cell) and C5 (400x300 cells, 5..400 ppc, ~20M particles: the two-array
    sort, dense-chunk fall-backs, embedded body, per-cell tau = tau_ref_n / N; PAPER.md:668 audits 8.0e6 particles on
    this grid)."""
    import torch
    tau_fn, kw = None, {}
    if case == "c3_4m":
        cfg, st = wl.cavity()
    elif case == "c4_8m":
        cfg, st = wl.cavity(n=200, ppc=200, kn=1.0, seed=42)
    else:
        cfg, st, _ = wl.cylinder()
        tau_ref_n = float(np.float32(cfg["tau"] * cfg["ppc_inf"]))
        tau_default = np.float32(cfg["tau"])

        def tau_fn(N):
            with np.errstate(divide="ignore", invalid="ignore"):
                return np.where(N > 0, np.float32(tau_ref_n) / np.maximum(N, 1).astype(np.float32), tau_default).astype(np.float32)
    ctx = gpu.Context(cfg)
    if tau_fn is not None:
        kw = dict(tau_mode=1, tau_ref_n=tau_ref_n, tau_cell=torch.empty(ctx.ncell, dtype=torch.float32, device="cuda"))
    a = gpu.to_device(st)
    b = {k: torch.empty_like(v) for k, v in a.items()}
    out = ctx.alloc_step_outputs(0)
    for it in range(3):                                  # a few steps so that counts are no longer the initial ones
        ctx.step(a, b, it, out, closure=0, **kw)
        a, b = b, a
    h = gpu.to_host(a)
    step_no = 3
    ctx.step(a, b, step_no, out, closure=0, **kw)
    got = gpu.to_host(b)
    res = {k: v.cpu().numpy() for k, v in out.items()}
    del a, b
    # oracle, stage by stage, each fed the GPU's own previous-stage output where floating point is involved
    s1 = orc.stream_walls(h, cfg, step_no)
    s2, cs, perm = orc.sort_by_cell(s1, cfg)
    assert np.array_equal(res["cell_start"], cs)
    assert np.array_equal(got["pid"], s2["pid"])
    assert np.array_equal(_bits(got["x"]), _bits(s2["x"])) and np.array_equal(_bits(got["y"]), _bits(s2["y"]))
    hit = _bits(s1["vx"]) != _bits(h["vx"])
    n = np.diff(cs)
    print("%s: %d particles, %d..%d per cell, %d wall / body re-emissions" % (case, h["x"].shape[0], n.min(), n.max(), int(hit.sum())))
    # moments of the oracle's sorted pre-update velocities (re-emitted ones differ from the GPU's by <= 1e-6)
    d2 = gpu.to_device(s2)
    cs_d = torch.from_numpy(cs).cuda()
    mom_g = ctx.cell_moments(d2["vx"], d2["vy"], d2["vz"], cs_d, 1).cpu().numpy()
    mom_o = orc.cell_moments(s2["vx"], s2["vy"], s2["vz"], cs, 1)
    rm = moment_ratio(mom_g, mom_o, absmom=abs_moments(s2["vx"], s2["vy"], s2["vz"], cs, mom_o))
    tau = cfg["tau"] if tau_fn is None else tau_fn(mom_o[:, 0])
    tau_d = None if tau_fn is None else torch.from_numpy(tau).cuda()
    coef_o, fl_o, kappa = orc.closure_exact(mom_o, tau, cfg["eps2_scale"], cfg["min_count"])
    coef_g, fl_g = ctx.closure_exact(torch.from_numpy(mom_o).cuda(), tau_d)
    hard = orc.FLAG_EMPTY | orc.FLAG_LOWCOUNT | orc.FLAG_SINGULAR
    assert np.array_equal(fl_g.cpu().numpy().view(np.uint32) & hard, fl_o & hard)
    ok = (fl_o & orc.FLAG_ILLCOND) == 0
    rc = coef_ratio(coef_g.cpu().numpy(), coef_o, tau, _theta(mom_o), 1e-5, mask=ok)
    c32 = coef_o.astype(np.float32)
    rvx, rvy, rvz, rfl = orc.velocity_update(s2["vx"], s2["vy"], s2["vz"], s2["pid"], cs, mom_o, c32, tau, cfg, step_no, fl_o)
    flg = torch.from_numpy(fl_o.view(np.int32).copy()).cuda()
    ctx.velocity_update(d2["vx"], d2["vy"], d2["vz"], d2["pid"], cs_d, torch.from_numpy(mom_o).cuda(),
                        torch.from_numpy(c32).cuda(), step_no, flg, tau_cell=tau_d)
    rv = velocity_ratio((d2["vx"].cpu().numpy(), d2["vy"].cpu().numpy(), d2["vz"].cpu().numpy()), (rvx, rvy, rvz), cs,
                        _theta(mom_o))
    print("%s full size: moments %.3f, closure %.3g (kappa max %.3g, %d ill-conditioned), update %.3f"
          % (case, rm, rc, kappa.max(), int((~ok).sum()), rv))
    assert rm <= 1.0 and rc <= 1.0 and rv <= 1.0
    assert np.array_equal(flg.cpu().numpy().view(np.uint32), rfl)
    for k in ("vx", "vy", "vz"):
        assert np.isfinite(got[k]).all()
    ctx.close()


# ------------------------------------------------------------------------------------------------ degenerate inputs
@pytest.mark.parametrize("n", [0, 1, 2, 3, 700])
@pytest.mark.parametrize("closure", [0, 1])
def test_step_degenerate_counts(gpu, wl, orc, n, closure):
    """No particle at all, fewer particles than the closure needs, and every particle in one cell of an otherwise
    empty grid (one 700-particle cell: the sliced path): the whole step must agree with the oracle, flags included."""
    import torch
    cfg = wl.make_config(6, 5, 1.0 / 6, 0.2, 0.01, 0.8, wl.NO_WALLS, seed=77, max_particles=max(n, 1))
    rng = np.random.default_rng(100 + n)
    st = {"x": (2.0 / 6 + rng.uniform(0.01, 0.15, n)).astype(np.float32), "y": (0.6 + rng.uniform(0.01, 0.18, n)).astype(np.float32),
          "vx": rng.normal(0.1, 0.7, n).astype(np.float32), "vy": rng.normal(0.0, 0.7, n).astype(np.float32),
          "vz": rng.normal(-0.2, 0.7, n).astype(np.float32), "pid": np.arange(n, dtype=np.uint32)}
    mlp = wl.xavier_mlp(seed=0, n_scale=1.0 / 60.0, tau=cfg["tau"], bias_scale=0.1) if closure else None
    got, res, ref, aux = _one_step(gpu, orc, cfg, st, closure, mlp, 3)
    assert np.array_equal(res["cell_start"], aux["cell_start"])
    assert np.array_equal(res["flags"].view(np.uint32), aux["flags"])
    for k in ("x", "y", "pid"):
        assert np.array_equal(_bits(got[k]), _bits(ref[k])), k
    occupied = aux["mom"][:, 0] > 0
    assert np.allclose(res["mom"][:, 0], aux["mom"][:, 0])
    if n:
        pre = _pre(orc, st, cfg, 3)
        r = moment_ratio(res["mom"], aux["mom"], absmom=abs_moments(pre[0], pre[1], pre[2], aux["cell_start"], aux["mom"]))
        assert r <= 1.0, r
        tol = 4e-6 if closure else 1e-6
        rv = velocity_ratio((got["vx"], got["vy"], got["vz"]), (ref["vx"], ref["vy"], ref["vz"]), aux["cell_start"],
                            _theta(aux["mom"]), tol=tol)
        assert rv <= 1.0, rv
    assert np.isfinite(res["coef"]).all()
    assert (res["coef"][~occupied] == 0).all()


def _pre(orc, st, cfg, step):
    """cell-sorted velocities before the update (what the moments were taken of)."""
    s2, _, _ = orc.sort_by_cell(orc.stream_walls(st, cfg, step), cfg)
    return s2["vx"], s2["vy"], s2["vz"]


# ------------------------------------------------------------------------------------------------ fallback paths
def test_unstaged_paths(gpu, wl, orc):
    """Per-warp staging needs 16-byte aligned arrays and cells that fit the warp's buffer.  Unaligned views and a
    cell of several thousand particles must take the global-memory path and still match the oracle."""
    import torch
    cfg, st = wl.ragged(nx=12, ny=9, seed=31, mean_ppc=70.0)
    # one huge cell: move 4000 extra particles into cell 17
    rng = np.random.default_rng(1)
    extra = 4000
    ex = {k: np.empty(extra, np.float32) for k in ("x", "y", "vx", "vy", "vz")}
    ex["x"][:] = (17 % 12 + rng.uniform(0.1, 0.9, extra)) / 12
    ex["y"][:] = (17 // 12 + rng.uniform(0.1, 0.9, extra)) / 9
    for k in ("vx", "vy", "vz"):
        ex[k][:] = rng.normal(0.2, 0.9, extra)
    st = {k: np.concatenate([st[k], ex[k]]) for k in ("x", "y", "vx", "vy", "vz")}
    st["pid"] = np.arange(st["x"].shape[0], dtype=np.uint32)
    cfg = dict(cfg, max_particles=int(st["x"].shape[0]) + 8)
    s, cs, _ = orc.sort_by_cell(st, cfg)
    n = s["x"].shape[0]
    ctx = gpu.Context(cfg)
    for off in (0, 1):          # off = 1: every array starts 4 bytes past a 16-byte boundary
        def dev(a, dt):
            buf = torch.empty(n + 4, dtype=dt, device="cuda")
            v = buf[off:off + n]
            v.copy_(torch.from_numpy(a.view(np.int32) if a.dtype == np.uint32 else a))
            return v
        vx, vy, vz = dev(s["vx"], torch.float32), dev(s["vy"], torch.float32), dev(s["vz"], torch.float32)
        pid = dev(s["pid"], torch.int32)
        csd = torch.from_numpy(cs).cuda()
        for mode in (0, 1):
            ref = orc.cell_moments(s["vx"], s["vy"], s["vz"], cs, mode)
            mom = ctx.cell_moments(vx, vy, vz, csd, mode)
            r = moment_ratio(mom.cpu().numpy(), ref, absmom=abs_moments(s["vx"], s["vy"], s["vz"], cs, ref))
            assert r <= 1.0, (off, mode, r)
        mom = orc.cell_moments(s["vx"], s["vy"], s["vz"], cs, 1)
        coef, flags, _ = orc.closure_exact(mom, cfg["tau"], cfg["eps2_scale"], cfg["min_count"])
        c32 = coef.astype(np.float32)
        rvx, rvy, rvz, rfl = orc.velocity_update(s["vx"], s["vy"], s["vz"], s["pid"], cs, mom, c32, cfg["tau"], cfg, 11, flags)
        fl = torch.from_numpy(flags.view(np.int32).copy()).cuda()
        ctx.velocity_update(vx, vy, vz, pid, csd, torch.from_numpy(mom).cuda(), torch.from_numpy(c32).cuda(), 11, fl)
        rv = velocity_ratio((vx.cpu().numpy(), vy.cpu().numpy(), vz.cpu().numpy()), (rvx, rvy, rvz), cs, _theta(mom))
        print("unstaged offset %d: update worst err/allowed %.3f" % (off, rv))
        assert rv <= 1.0
        assert np.array_equal(fl.cpu().numpy().view(np.uint32), rfl)
    ctx.close()
