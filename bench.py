#!/usr/bin/env python
"""bench.py -- throughput of the cubic-FP closure hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl fpcl|reference] [--closure exact|mlp] [--small]

One "step" = one fp_step (stream -> walls -> sort -> moment gather -> closure -> velocity update) over the
BASELINE config-3 ensemble: 2D lid-driven cavity, 200x200 cells x 100 particles/cell = 4M particles, synthetic
(seeded Maxwellian, 200 settling steps before timing so that cell counts are Poisson-like).  `value` is
particle-steps/s with all inputs resident in HBM; `e2e` is the same metric through fp_step_host (pinned host
buffers, H2D + D2H inside the timed region).  Multi-GPU (torchrun): every rank runs an independent replica with its
own seed (weak scaling, no data-path collective -- DESIGN.md "Multi-GPU"); times are max-reduced over ranks.

--impl reference times the CPU oracle (oracle/, plain C fp64, as it stands) on the host cores on a bounded sample
of the same workload; it is a deliberately slow checker, not a competitor.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle_steps_per_s"
UNIT = "particle-steps/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="fpcl", choices=["fpcl", "reference"])
    ap.add_argument("--closure", default="exact", choices=["exact", "mlp"])
    ap.add_argument("--settle", type=int, default=200, help="untimed steps that relax the initial uniform counts")
    ap.add_argument("--small", action="store_true", help="64x64x100 cavity (debugging only; not a bench line)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the cold-L2 kernel table and the MLP variant")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def workload(args, seed):
    from paper_2606_15622_b200 import workloads
    n = 64 if args.small else 200
    cfg, st = workloads.cavity(n=n, ppc=100, kn=0.5, seed=seed, shuffle=True)
    name = "cavity Kn=0.5 %dx%d cells x 100 ppc = %d particles (BASELINE config 3%s)" % (
        n, n, st["x"].shape[0], ", reduced" if args.small else "")
    return cfg, st, name


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 20 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [v.strip() for v in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_model():
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample(cfg, st, closure, mlp, max_seconds=12.0, max_steps=10, threads=1):
    """The oracle as it stands (fp64) stepping the same ensemble with `threads` OpenMP threads (0 = all cores) in its
    per-cell / per-particle loops; returns (particle-steps/s, steps, seconds, threads used)."""
    import oracle
    oracle.build()
    used = oracle.set_threads(threads)
    s = {k: v.copy() for k, v in st.items()}
    n = s["x"].shape[0]
    t0 = time.perf_counter()
    done = 0
    while done < max_steps:
        s, _ = oracle.step(s, cfg, done, closure=closure, mlp=mlp)
        done += 1
        if time.perf_counter() - t0 > max_seconds:
            break
    dt = time.perf_counter() - t0
    return n * done / dt, done, dt, used


def run_reference(args):
    """--impl reference: the oracle on the host cores, same config / metric / unit (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2606_15622_b200 import workloads
    cfg, st, name = workload(args, seed=3)
    mlp = workloads.xavier_mlp(n_scale=0.01, tau=cfg["tau"]) if args.closure == "mlp" else None
    n = st["x"].shape[0]
    # each "step" of this arm is one oracle step on a bounded sample: the first n_s particles' worth of cells
    rows = 20 if not args.small else 8                      # 20 of 200 cell rows = 400k particles per step
    ny = cfg["ny"]
    keep = st["y"] < (rows / ny)
    sub = {k: np.ascontiguousarray(v[keep]) for k, v in st.items()}
    scfg = dict(cfg, ny=rows, max_particles=int(keep.sum()))
    import oracle
    oracle.build()
    used = oracle.set_threads(0)
    s = sub
    for w in range(min(args.warmup, 1)):
        s, _ = oracle.step(s, scfg, w, closure=args.closure, mlp=mlp)
    t0 = time.perf_counter()
    for k in range(args.steps):
        s, _ = oracle.step(s, scfg, 100 + k, closure=args.closure, mlp=mlp)
    dt = time.perf_counter() - t0
    val = s["x"].shape[0] * args.steps / dt
    sample = "%d oracle steps on a %dx%d-cell slab of the cavity (%d particles), %d threads (%s)" % (
        args.steps, cfg["nx"], rows, s["x"].shape[0], used, cpu_model())
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "closure": args.closure, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def algorithmic_bytes(np_, ncell):
    """Algorithmic HBM bytes per launch."""
    return {
        "stream_walls": 28 * np_,                          # 16 r (x,y,vx,vy) + 8 w (x,y) + 4 w key
        "moments_full": 12 * np_ + 236 * ncell,            # 12 B/particle + cell_start + 232 B record
        "moments_lite": 12 * np_ + 108 * ncell,
        "closure_exact": 272 * ncell,                      # 232 r + 36 w + 4 w flags
        "closure_mlp": 144 * ncell,                        # 104 r + 36 w + 4 w
        "update": 28 * np_ + (4 + 232 + 36 + 4) * ncell,   # 12 r + 4 r pid + 12 w; per cell start, record, coef, flags
        "update_lite": 28 * np_ + (4 + 104 + 36 + 4) * ncell,
        "cell_diagnostics": (232 + 128) * ncell,           # FULL record read, 16 doubles written (NEXT-2)
        "gather": 52 * np_,                                # 4 r perm + 24 r + 24 w
        "sort_keys": 36 * np_,                             # 2 passes x (4+4 r hist+scatter keys) + idx r/w
    }


def cold_kernel_table(fpcl, torch, ctx, state, out, mlp_dev, hbm_peak, reps=20):
    """Stand-alone launches of the judged kernels with an L2 flush (256 MB write) before each timed launch."""
    np_ = state["x"].numel()
    ncell = ctx.ncell
    ab = algorithmic_bytes(np_, ncell)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")
    cs = out["cell_start"]
    mom_full = torch.empty((ncell, 29), dtype=torch.float64, device="cuda")
    mom_lite = torch.empty((ncell, 13), dtype=torch.float64, device="cuda")
    coef = torch.zeros((ncell, 9), dtype=torch.float32, device="cuda")
    flags = torch.zeros(ncell, dtype=torch.int32, device="cuda")
    v = [state[k].clone() for k in ("vx", "vy", "vz")]
    ctx.cell_moments(v[0], v[1], v[2], cs, 1, out=mom_full)
    ctx.cell_moments(v[0], v[1], v[2], cs, 0, out=mom_lite)
    fpcl.fp_closure_exact(ctx.h, mom_full, None, coef, flags)

    def timed(fn, key):
        ts = []
        for r in range(reps + 3):
            flush.fill_(float(r))
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn(r)
            e1.record()
            e1.synchronize()
            if r >= 3:
                ts.append(e0.elapsed_time(e1))
        ms = float(np.median(ts))
        gbs = ab[key] / (ms * 1e-3) / 1e9
        return {"ms": ms, "best_ms": float(min(ts)), "GBps": gbs, "frac_of_hbm_peak": gbs / hbm_peak,
                "algorithmic_bytes": ab[key]}

    res = {}
    res["moments_full"] = timed(lambda r: ctx.cell_moments(v[0], v[1], v[2], cs, 1, out=mom_full), "moments_full")
    res["moments_lite"] = timed(lambda r: ctx.cell_moments(v[0], v[1], v[2], cs, 0, out=mom_lite), "moments_lite")
    res["closure_exact"] = timed(lambda r: fpcl.fp_closure_exact(ctx.h, mom_full, None, coef, flags), "closure_exact")
    res["closure_exact"]["cells_per_s"] = ncell / (res["closure_exact"]["ms"] * 1e-3)
    diag = torch.empty((ncell, 16), dtype=torch.float64, device="cuda")
    res["cell_diagnostics"] = timed(lambda r: ctx.cell_diagnostics(mom_full, 0.5, 100.0, 0.0, out=diag), "cell_diagnostics")
    res["cell_diagnostics"]["cells_per_s"] = ncell / (res["cell_diagnostics"]["ms"] * 1e-3)
    if mlp_dev is not None:
        res["closure_mlp"] = timed(lambda r: fpcl.fp_closure_mlp(ctx.h, mom_lite, 13, None, mlp_dev, 1.0, coef, flags),
                                   "closure_mlp")
        res["closure_mlp"]["cells_per_s"] = ncell / (res["closure_mlp"]["ms"] * 1e-3)
        res["closure_mlp"]["kernel"] = "mma.sync TF32 with 3xTF32 compensation (default, ~1e-5)"
    fpcl.fp_closure_exact(ctx.h, mom_full, None, coef, flags)
    # the update rewrites velocities in place: each timed launch advances the same ensemble one collision step
    ts = []
    for r in range(reps + 3):
        ctx.cell_moments(v[0], v[1], v[2], cs, 1, out=mom_full)      # moments of the current velocities (untimed)
        flush.fill_(float(r))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.velocity_update(v[0], v[1], v[2], state["pid"], cs, mom_full, coef, 1000 + r, flags)
        e1.record()
        e1.synchronize()
        if r >= 3:
            ts.append(e0.elapsed_time(e1))
    ms = float(np.median(ts))
    gbs = ab["update"] / (ms * 1e-3) / 1e9
    res["update"] = {"ms": ms, "best_ms": float(min(ts)), "GBps": gbs, "frac_of_hbm_peak": gbs / hbm_peak,
                     "algorithmic_bytes": ab["update"], "particles_per_s": np_ / (ms * 1e-3)}
    res["moments_full"]["particles_per_s"] = np_ / (res["moments_full"]["ms"] * 1e-3)
    # Second cold-L2 protocol (SURVEY 8(d) "rotate over >= 4 independent copies"): back-to-back launches over
    # independent copies of the particle arrays whose footprint is >= 2.5x the 126 MB L2, one event pair around the
    # whole batch.  No flush kernel and no per-launch event pair inside the timed region, so the ~4 us of launch
    # latency and event granularity that a single ~25 us launch carries above is amortised away.
    ncopy = int(max(4, min(12, -(-320e6 // (12 * np_)))))
    vc = [[t.clone() for t in v] for _ in range(ncopy)]
    pidc = [state["pid"].clone() for _ in range(ncopy)]
    momc = [torch.empty_like(mom_full) for _ in range(ncopy)]

    def batch(fn, rounds=4, before=None):
        for c in range(ncopy):
            fn(c, -1)
        tot = 0.0
        for r in range(rounds):
            if before is not None:
                before()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for c in range(ncopy):
                fn(c, r)
            e1.record()
            e1.synchronize()
            tot += e0.elapsed_time(e1)
        return tot / (rounds * ncopy)

    def add_rot(key, ms):
        gbs = ab[key] / (ms * 1e-3) / 1e9
        res[key].update({"ms_rotating": ms, "GBps_rotating": gbs, "frac_of_hbm_peak_rotating": gbs / hbm_peak,
                         "rotating_copies": ncopy})

    add_rot("moments_full", batch(lambda c, r: ctx.cell_moments(vc[c][0], vc[c][1], vc[c][2], cs, 1, out=mom_full)))
    add_rot("moments_lite", batch(lambda c, r: ctx.cell_moments(vc[c][0], vc[c][1], vc[c][2], cs, 0, out=mom_lite)))

    def fresh_moments():
        for c in range(ncopy):
            ctx.cell_moments(vc[c][0], vc[c][1], vc[c][2], cs, 1, out=momc[c])

    fresh_moments()
    add_rot("update", batch(lambda c, r: ctx.velocity_update(vc[c][0], vc[c][1], vc[c][2], pidc[c], cs, momc[c], coef,
                                                              2000 + r, flags), before=fresh_moments))
    res["protocols"] = ("ms: 256 MB L2-flushing write, then one launch between its own event pair (median); "
                        "ms_rotating: back-to-back launches over %d independent copies of the particle arrays "
                        "(%.0f MB), one event pair per batch" % (ncopy, ncopy * 12 * np_ / 1e6))
    return res


def judged_kernels_cold(fpcl, torch, ctx, state, out, hbm_peak, rounds=4):
    """The two kernels north_star judges (moment gather, velocity update) stand-alone with a cold L2: back-to-back
    launches over independent copies of the particle arrays whose footprint is >= 2.5x the 126 MB L2, one CUDA event
    pair around each batch (SURVEY 8(d) 'rotate over >= 4 independent copies').  fp_velocity_update as a user calls
    it, i.e. including its per-cell constants kernel.  Part of every bench line (about one second)."""
    np_, ncell = state["x"].numel(), ctx.ncell
    ab = algorithmic_bytes(np_, ncell)
    cs = out["cell_start"]
    ncopy = int(max(4, min(12, -(-320e6 // (12 * np_)))))
    vc = [[state[k].clone() for k in ("vx", "vy", "vz")] for _ in range(ncopy)]
    pidc = [state["pid"].clone() for _ in range(ncopy)]
    mom_full = torch.empty((ncell, 29), dtype=torch.float64, device="cuda")
    mom_lite = torch.empty((ncell, 13), dtype=torch.float64, device="cuda")
    momc = [torch.empty_like(mom_full) for _ in range(ncopy)]
    coef = torch.zeros((ncell, 9), dtype=torch.float32, device="cuda")
    flags = torch.zeros(ncell, dtype=torch.int32, device="cuda")
    ctx.cell_moments(vc[0][0], vc[0][1], vc[0][2], cs, 1, out=mom_full)
    fpcl.fp_closure_exact(ctx.h, mom_full, None, coef, flags)

    def batch(fn, before=None):
        for c in range(ncopy):
            fn(c, -1)
        best = float("inf")
        for r in range(rounds):
            if before is not None:
                before()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for c in range(ncopy):
                fn(c, r)
            e1.record()
            e1.synchronize()
            best = min(best, e0.elapsed_time(e1) / ncopy)
        return best

    def entry(key, ms):
        gbs = ab[key] / (ms * 1e-3) / 1e9
        return {"ms": ms, "GBps": gbs, "frac": gbs / hbm_peak, "algorithmic_bytes": ab[key]}

    def fresh_moments():
        for c in range(ncopy):
            ctx.cell_moments(vc[c][0], vc[c][1], vc[c][2], cs, 1, out=momc[c])

    res = {"moments_full": entry("moments_full", batch(lambda c, r: ctx.cell_moments(vc[c][0], vc[c][1], vc[c][2], cs, 1, out=mom_full))),
           "moments_lite": entry("moments_lite", batch(lambda c, r: ctx.cell_moments(vc[c][0], vc[c][1], vc[c][2], cs, 0, out=mom_lite)))}
    fresh_moments()
    res["update"] = entry("update", batch(lambda c, r: ctx.velocity_update(vc[c][0], vc[c][1], vc[c][2], pidc[c], cs, momc[c], coef,
                                                                         3000 + r, flags), before=fresh_moments))
    res["protocol"] = ("cold-L2 rotating: back-to-back launches over %d independent copies of the particle arrays (%.0f MB), "
                       "one event pair per batch, best of %d batches" % (ncopy, ncopy * 12 * np_ / 1e6, rounds))
    return res


def committed_traffic(kernel_source):
    """DRAM bytes per launch of the judged kernels from the committed ncu --set full capture (profiles/r02_traffic.csv:
    kernel, dram_bytes, source file, sha256 of that source at capture time).  A row whose source has changed since is
    stale and is not reported."""
    import csv
    import hashlib
    out = {}
    path = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    if not os.path.exists(path):
        return out
    for row in csv.DictReader(open(path)):
        src = os.path.join(ROOT, row["source"])
        if os.path.exists(src) and hashlib.sha256(open(src, "rb").read()).hexdigest()[:16] == row["sha256_16"]:
            out[row["kernel"]] = float(row["dram_bytes"])
    return out


def paper_surrogate(fpcl, torch, workloads, tau):
    """the paper's own surrogate (16 features -> 4 x 256 ReLU -> 9) with
    under-relaxation w = 0.2 (:568), on LITE records of C3-sized (40k cells) and C5-sized (120k cells) grids.
    Tensor-core kernel (mlp_wide.cuh): split-bf16 products, three mma per useful product."""
    bf16_peak, src = 2250.0, "nominal dense bf16 (B200_PROFILING.md)"
    try:
        bf16_peak, src = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["bf16_tflops"]), "measured cuBLAS bf16 (MEASURED_PEAKS.json)"
    except Exception:
        pass
    dims = (16, 256, 256, 256, 256, 9)
    mac = sum(dims[i] * dims[i + 1] for i in range(len(dims) - 1))
    res = {"network": "16-256-256-256-256-9 ReLU, %d parameters, relax_w = 0.2" % (mac + sum(dims[1:])),
           "kernels": {"tcgen05": "mlp_wide5_kernel: tcgen05.mma cta_group::1 kind::f16 (bf16), M 128 x N 256 x K 16, accumulator "
                                  "in TMEM, 3 split products per useful product (~2.8e-5 of the output scale vs the oracle)",
                       "mma_sync": "mlp_wide_kernel: mma.sync m16n8k16 bf16, same arithmetic (fp_set_mlp_tensor_cores(ctx, 2))"},
           "peak_source": src}
    mlp = fpcl.Mlp(workloads.xavier_mlp(dims=dims, seed=0, act=1, feature_set=1, n_scale=0.05, tau=tau))
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")
    for name, n in (("cells_40000", 200), ("cells_119716", 346)):
        cfg, _ = workloads.cavity(n=n, ppc=30, kn=0.5, seed=3, shuffle=False)
        ctx = fpcl.Context(cfg)
        ncell = ctx.ncell
        g = torch.Generator(device="cuda"); g.manual_seed(11)
        cnt = torch.poisson(torch.full((ncell,), 20.0, device="cuda"), generator=g).to(torch.int32)
        cs = torch.zeros(ncell + 1, dtype=torch.int32, device="cuda"); cs[1:] = torch.cumsum(cnt, 0)
        npart = int(cs[-1])
        v = [(torch.randn(npart, device="cuda", generator=g) * 0.7071).contiguous() for _ in range(3)]
        mom = ctx.cell_moments(v[0], v[1], v[2], cs, 0)
        coef = torch.zeros((ncell, 9), dtype=torch.float32, device="cuda")
        flags = torch.zeros(ncell, dtype=torch.int32, device="cuda")
        entry = {}
        for kname, mode in (("tcgen05", 1), ("mma_sync", 2)):
            fpcl.fp_set_mlp_tensor_cores(ctx.h, mode)
            ts = []
            for r in range(13):
                flush.fill_(float(r))
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                fpcl.fp_closure_mlp(ctx.h, mom, 13, None, mlp, 0.2, coef, flags)
                e1.record(); e1.synchronize()
                if r >= 3:
                    ts.append(e0.elapsed_time(e1))
            ms = float(np.median(ts))
            useful = 2.0 * mac * ncell / (ms * 1e-3) / 1e12
            entry[kname] = {"ms": ms, "cells_per_s": ncell / (ms * 1e-3), "useful_TFLOPs": useful,
                            "roofline": {"bound": "tensor", "achieved": 3.0 * useful, "peak": bf16_peak, "unit": "TFLOP/s",
                                         "frac": 3.0 * useful / bf16_peak,
                                         "note": "achieved counts the three bf16 products executed per useful product"},
                            "flagged_cells": int((flags != 0).sum().item())}
        res[name] = entry
        ctx.close()
        del v, mom, coef, flags
    return res


def couette_small(fpcl, torch, workloads):
    """BASELINE config 1: 1D Couette, 50 cells x 100 particles, 100 fp_steps with the exact closure and again with the
    13-64-64-64-9 SiLU surrogate.  At 5,000 particles a step is nine kernel launches' worth of latency."""
    res = {}
    cfg, st = workloads.couette()
    mlp = fpcl.Mlp(workloads.xavier_mlp(n_scale=0.01, tau=cfg["tau"]))
    for name, closure in (("exact", 0), ("mlp", 1)):
        ctx = fpcl.Context(cfg)
        a = fpcl.to_device(st)
        b = {k: torch.empty_like(v) for k, v in a.items()}
        out = ctx.alloc_step_outputs(closure)
        for w in range(10):
            ctx.step(a, b, w, out, closure=closure, mlp=mlp if closure else None); a, b = b, a
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for w in range(100):
            ctx.step(a, b, 10 + w, out, closure=closure, mlp=mlp if closure else None); a, b = b, a
        e1.record(); e1.synchronize()
        ms = e0.elapsed_time(e1) / 100
        res[name] = {"particles": int(a["x"].numel()), "cells": ctx.ncell, "ms_per_step": ms,
                     "particle_steps_per_s": a["x"].numel() / (ms * 1e-3),
                     "flagged_cells": int((out["flags"] != 0).sum().item())}
        ctx.close()
    return res


def closure_microbench(fpcl, torch, workloads, mlp_dev, hbm_peak):
    """BASELINE config 2: 100x100 cells x 50 particles from a Grad-13-perturbed Maxwellian (seed 1), no streaming:
    moment gather, exact closure and surrogate timed separately (cold L2), flag counts and a histogram of the exact
    closure's condition estimates.  With |s_ij| <= 0.3, |q| <= 0.2 and 50 particles per cell this recipe stays well
    conditioned (kappa_1 <= ~1e2 with the eps^2 term of reading R2-e); the ill-conditioned half of the closure contract
    (kappa up to 1e16, singular cells) is exercised by tests/test_gpu_parity.py::test_closure_exact_conditioning."""
    cfg, st = workloads.grad13_cells()[:2]
    ctx = fpcl.Context(cfg)
    srt, cs, _ = ctx.sort_by_cell(fpcl.to_device(st), want_perm=False)
    out = {"cell_start": cs}
    tab = cold_kernel_table(fpcl, torch, ctx, srt, out, mlp_dev, hbm_peak, reps=20)
    mom = ctx.cell_moments(srt["vx"], srt["vy"], srt["vz"], cs, 1)
    coef, flags, kappa = ctx.closure_exact(mom, want_kappa=True)
    kap = kappa.cpu().numpy()
    fl = flags.cpu().numpy().view(np.uint32)
    edges = [0.0, 10.0, 20.0, 40.0, 80.0, 160.0, 1e3, 1e4, 1e6, 1e8, float("inf")]
    hist, _ = np.histogram(kap[kap > 0], bins=edges)
    res = {"particles": int(srt["x"].numel()), "cells": ctx.ncell, "kernels_cold_l2": tab,
           "flag_counts": {"illcond": int((fl & 8 != 0).sum()), "singular": int((fl & 4 != 0).sum()),
                           "lowcount": int((fl & 2 != 0).sum()), "empty": int((fl & 1 != 0).sum())},
           "kappa_estimate_histogram": {"edges": edges[:-1] + ["inf"], "counts": [int(c) for c in hist]}}
    ctx.close()
    return res


def ppc_sweep(fpcl, torch, workloads, n_steps, steps_20ppc=None):
    """BASELINE config 4: cavity Kn = 1.0, 200x200 cells, 20 / 50 / 200 particles per cell (seeds 40/41/42), n_steps
    fp_steps with the exact closure.  Reports throughput and the conservation drift of the collision step: every
    100th step the per-cell mean velocity and energy after the update (a second moment pass over the updated
    velocities; the update moves no particle between cells) are compared with the moments the step itself took before
    the update.  Scales: sqrt(theta) for the mean, 3 theta for the energy; cells the update skips are excluded."""
    res = {}
    n_default = n_steps
    for ppc, seed in ((20, 40), (50, 41), (200, 42)):
        # BASELINE config 4 asks for the drift after 1,000 steps: the 20-ppc case (74 us per step) always runs them
        n_steps = steps_20ppc if (ppc == 20 and steps_20ppc) else n_default
        cfg, st = workloads.cavity(n=200, ppc=ppc, kn=1.0, seed=seed, shuffle=True)
        ctx = fpcl.Context(cfg)
        a = fpcl.to_device(st)
        b = {k: torch.empty_like(v) for k, v in a.items()}
        out = ctx.alloc_step_outputs(0)
        np_ = a["x"].numel()
        after = torch.empty((ctx.ncell, 13), dtype=torch.float64, device="cuda")
        dmom, dene, flagged, nonfinite = 0.0, 0.0, 0, 0
        energy = []
        for w in range(5):
            ctx.step(a, b, w, out, closure=0); a, b = b, a
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ms = 0.0
        for blk in range(0, n_steps, 100):
            nb = min(100, n_steps - blk)
            e0.record()
            for k in range(nb):
                ctx.step(a, b, 5 + blk + k, out, closure=0); a, b = b, a
            e1.record(); e1.synchronize()
            ms += e0.elapsed_time(e1)
            # drift of the last step of the block (a now holds its output)
            ctx.cell_moments(a["vx"], a["vy"], a["vz"], out["cell_start"], 0, out=after)
            before = out["mom"]
            n = before[:, 0]
            theta = (before[:, 4] + before[:, 7] + before[:, 9]) / 3.0
            act = (n >= 2) & (theta > 0) & ((out["flags"] & 32) == 0)
            if bool(act.any()):
                du = (after[:, 1:4] - before[:, 1:4]).abs().amax(dim=1) / theta.clamp_min(1e-300).sqrt()
                de = ((after[:, 4] + after[:, 7] + after[:, 9]) - 3.0 * theta).abs() / (3.0 * theta.clamp_min(1e-300))
                dmom = max(dmom, float(du[act].max().item()))
                dene = max(dene, float(de[act].max().item()))
            flagged = max(flagged, int((out["flags"] != 0).sum().item()))
            v2 = a["vx"].double() ** 2 + a["vy"].double() ** 2 + a["vz"].double() ** 2
            nonfinite += int((~torch.isfinite(v2)).sum().item())
            energy.append(float(v2.sum().item()) / np_)
        res["ppc_%d" % ppc] = {"particles": np_, "steps": n_steps, "ms_per_step": ms / n_steps,
                               "particle_steps_per_s": np_ * n_steps / (ms * 1e-3),
                               "delta_particles": int(a["x"].numel() - np_),
                               "collision_step_max_rel_momentum_change": dmom,
                               "collision_step_max_rel_energy_change": dene,
                               "max_flagged_cells": flagged, "nonfinite_velocities": nonfinite,
                               "mean_v2_per_particle_every_100_steps": energy}
        ctx.close()
        del a, b, out, after
        torch.cuda.empty_cache()
    return res


def corroborate(fpcl, torch, workloads, mlp_dev, hbm_peak, steps):
    """the judged kernels again where the velocity arrays cannot sit in the 126 MB L2 -- C4 at 200 ppc
    (8M particles, 96 MB of velocities) and C5 (hypersonic cylinder, ~20M particles, 5..400 per cell, 240 MB)."""
    res = {}
    for name in ("c4_8m", "c5"):
        if name == "c4_8m":
            cfg, st = workloads.cavity(n=200, ppc=200, kn=1.0, seed=42, shuffle=True)
            kw = {}
            label = "cavity Kn=1.0 200x200 cells x 200 ppc (BASELINE config 4)"
        else:
            cfg, st, _tau = workloads.cylinder()
            tau_buf = torch.empty(cfg["nx"] * cfg["ny"], dtype=torch.float32, device="cuda")
            kw = dict(tau_mode=1, tau_ref_n=cfg["tau"] * cfg["ppc_inf"], tau_cell=tau_buf)
            label = "hypersonic cylinder 400x300 cells, 5..400 ppc (BASELINE config 5)"
        ctx = fpcl.Context(cfg)
        a = fpcl.to_device(st)
        b = {k: torch.empty_like(v) for k, v in a.items()}
        out = ctx.alloc_step_outputs(0)
        # C5's outer faces are a freestream reservoir (FP_WALL_INFLOW, R11): the particle count is constant and the
        # loop is closed, so it is stepped like the others (the analytic bow-shock field it starts from is not a steady
        # solution: the flow keeps evolving, the report says what the cell populations look like when it is timed)
        warm, steps_here = (10, steps) if name == "c4_8m" else (100, steps)
        n = 0
        for _ in range(warm):
            ctx.step(a, b, n, out, closure=0, **kw); a, b = b, a; n += 1
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps_here):
            ctx.step(a, b, n, out, closure=0, **kw); a, b = b, a; n += 1
        e1.record(); e1.synchronize()
        np_ = a["x"].numel()
        ms = e0.elapsed_time(e1) / steps_here
        tab = cold_kernel_table(fpcl, torch, ctx, a, out, mlp_dev, hbm_peak, reps=8)
        counts = (out["cell_start"][1:] - out["cell_start"][:-1])
        res[name] = {"workload": label, "particles": np_, "cells": ctx.ncell, "fp_step_ms": ms, "steps": steps_here,
                     "max_particles_per_cell": int(counts.max().item()),
                     "particles_per_cell_percentiles_50_99_99.9": [int(v) for v in torch.quantile(
                         counts[counts > 0].float()[:: max(1, int(counts.numel()) // 100000)], torch.tensor([0.5, 0.99, 0.999], device="cuda")).tolist()],
                     "warmup_steps": warm,
                     "particle_steps_per_s": np_ / (ms * 1e-3),
                     "flags_nonzero_cells": int((out["flags"] != 0).sum().item()), "kernels_cold_l2": tab}
        ctx.close()
        del a, b, out
        torch.cuda.empty_cache()
    return res


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    from paper_2606_15622_b200 import dist as D, fpcl, workloads

    world, rank, local = D.world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    D.init("nccl", torch.device("cuda", local))
    hbm_peak, peak_src = peaks()
    closure = 0 if args.closure == "exact" else 1

    # independent replica per rank: same shape, different seed (weak scaling)
    cfg, st, wname = workload(args, seed=D.replica_seed(3, rank))
    np_ = st["x"].shape[0]
    ncell = cfg["nx"] * cfg["ny"]
    mlp_host = workloads.xavier_mlp(n_scale=0.01, tau=cfg["tau"])
    mlp_dev = fpcl.Mlp(mlp_host)
    ctx = fpcl.Context(cfg)
    a = fpcl.to_device(st)
    b = {k: torch.empty_like(v) for k, v in a.items()}
    out = ctx.alloc_step_outputs(closure)
    step_no = 0
    for _ in range(args.settle):
        ctx.step(a, b, step_no, out, closure=closure, mlp=mlp_dev if closure else None)
        a, b = b, a
        step_no += 1
    torch.cuda.synchronize()
    settled = fpcl.to_host(a)                     # host copy of the settled ensemble: e2e and oracle input

    def barrier():
        D.barrier()
        torch.cuda.synchronize()

    # ---- timed region: K fp_step calls, device-resident
    for _ in range(args.warmup):
        ctx.step(a, b, step_no, out, closure=closure, mlp=mlp_dev if closure else None)
        a, b = b, a
        step_no += 1
    l0 = fpcl.fp_launch_count(ctx.h)
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        ctx.step(a, b, step_no, out, closure=closure, mlp=mlp_dev if closure else None)
        a, b = b, a
        step_no += 1
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = e0.elapsed_time(e1)
    launches = fpcl.fp_launch_count(ctx.h) - l0
    # ---- the same K steps again with the library's per-stage CUDA events switched on (seven event records per
    # step sit between the kernels and cost a few microseconds each, so the headline above is timed without them)
    fpcl.fp_timing_enable(ctx.h, args.steps)
    barrier()
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2.record()
    for _ in range(args.steps):
        ctx.step(a, b, step_no, out, closure=closure, mlp=mlp_dev if closure else None)
        a, b = b, a
        step_no += 1
    e3.record()
    barrier()
    ms_total_staged = e2.elapsed_time(e3)
    stage_ms = fpcl.fp_timing_read(ctx.h, args.steps)
    fpcl.fp_timing_enable(ctx.h, 0)
    ms_total = D.max_over_ranks(ms_total, "cuda")
    value = D.aggregate_throughput(np_, args.steps, ms_total, world)
    flags_host = out["flags"].cpu().numpy().view(np.uint32)

    # ---- end to end through fp_step_host: pinned host buffers, H2D + D2H inside the timed region
    pinned = {k: torch.from_numpy(v.view(np.int32) if k == "pid" else v).pin_memory() for k, v in settled.items()}
    hc = torch.empty((ncell, 9), dtype=torch.float32).pin_memory()
    hf = torch.empty(ncell, dtype=torch.int32).pin_memory()
    hs = torch.empty(ncell + 1, dtype=torch.int32).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    for w in range(2):
        ctx.step_host(pinned, 10_000 + w, closure=closure, mlp=mlp_dev if closure else None, h_coef=hc, h_flags=hf,
                      h_cell_start=hs)
    barrier()
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        ctx.step_host(pinned, 20_000 + k, closure=closure, mlp=mlp_dev if closure else None, h_coef=hc, h_flags=hf,
                      h_cell_start=hs)
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_value = D.aggregate_throughput(np_, e2e_steps, 1e3 * D.max_over_ranks(e2e_s, "cuda"), world)
    h2d = 24 * np_
    d2h = 24 * np_ + ncell * (36 + 4) + (ncell + 1) * 4

    # ---- per-stage times inside the timed region (CUDA events recorded by the library on the launch stream)
    ab = algorithmic_bytes(np_, ncell)
    med = np.median(stage_ms, axis=0) if stage_ms.shape[0] else np.zeros(fpcl.NSTAGES)
    stage_bytes = [ab["stream_walls"], ab["sort_keys"], ab["gather"], ab["moments_full" if closure == 0 else "moments_lite"],
                   ab["closure_exact" if closure == 0 else "closure_mlp"], ab["update" if closure == 0 else "update_lite"]]
    stages = {}
    for k, nme in enumerate(fpcl.STAGE_NAMES):
        gbs = stage_bytes[k] / (med[k] * 1e-3) / 1e9 if med[k] > 0 else 0.0
        stages[nme] = {"ms": float(med[k]), "share": float(med[k] / med.sum()) if med.sum() > 0 else 0.0,
                       "GBps_algorithmic": gbs, "frac_of_hbm_peak": gbs / hbm_peak}
    # roofline: the judged numbers are the cold-L2 stand-alone launches of the moment gather and the velocity update
    # (north_star: each >= 60 % of HBM roofline at C3); the headline object is the larger of the two kernels (update),
    # the other one and the in-step (L2-warm) stage figures ride along under "also"
    single = {n: stages[n] for n in ("stream_walls", "gather", "moments", "closure", "update")}
    dom = max(single, key=lambda n: single[n]["ms"])
    cold = judged_kernels_cold(fpcl, torch, ctx, a, out, hbm_peak) if rank == 0 else None
    roofline = None
    if cold is not None:
        traffic = committed_traffic("update") if not args.small else {}
        roofline = {"kernel": "update (fp_velocity_update, stand-alone)", "bound": "hbm", "achieved": cold["update"]["GBps"],
                    "peak": hbm_peak, "unit": "GB/s", "frac": cold["update"]["frac"], "traffic": traffic.get("update"),
                    "peak_source": peak_src, "timing": cold["protocol"], "ms": cold["update"]["ms"],
                    "also": {"moments_full": dict(cold["moments_full"], traffic=traffic.get("moments_full")),
                             "moments_lite": dict(cold["moments_lite"], traffic=traffic.get("moments_lite")),
                             "update_in_step_l2_warm": {"ms": single["update"]["ms"], "GBps": single["update"]["GBps_algorithmic"],
                                                        "frac": single["update"]["frac_of_hbm_peak"]},
                             "moments_in_step_l2_warm": {"ms": single["moments"]["ms"], "GBps": single["moments"]["GBps_algorithmic"],
                                                         "frac": single["moments"]["frac_of_hbm_peak"]},
                             "dominant_kernel_in_step": {"kernel": dom, "ms": single[dom]["ms"],
                                                         "frac": single[dom]["frac_of_hbm_peak"]}}}
        # the update kernel against its own bound ("What bounds it: the FMA pipe"): the pass-A loop
        # needs 446 scheduler cycles per 64 particles (measured in isolation), a B200 has 148 x 4 schedulers
        sm_hz = 1e6 * float(clocks.get("sm_mhz") or 1965.0)
        sms = torch.cuda.get_device_properties(0).multi_processor_count
        need = 446.0 / 64.0 * np_ / (cold["update"]["ms"] * 1e-3)
        roofline["also"]["update_alu"] = {"bound": "alu", "unit": "scheduler-cycles/s", "achieved": need,
                                          "peak": sms * 4 * sm_hz, "frac": need / (sms * 4 * sm_hz),
                                          "peak_source": "SMs x 4 schedulers x SM clock under load",
                                          "note": "pass A only: Philox4x32-10 + Box-Muller + cubic drift per particle"}

    extras = {}
    if rank == 0 and not args.no_extras:
        extras["kernels_cold_l2"] = cold_kernel_table(fpcl, torch, ctx, a, out, mlp_dev, hbm_peak)
        # the surrogate variant of the whole step (Algorithm 2), short run
        out2 = ctx.alloc_step_outputs(1)
        a2 = {k: v.clone() for k, v in a.items()}
        b2 = {k: torch.empty_like(v) for k, v in a.items()}
        for w in range(3):
            ctx.step(a2, b2, 50_000 + w, out2, closure=1, mlp=mlp_dev); a2, b2 = b2, a2
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record()
        nrep = min(args.steps, 20)
        for w in range(nrep):
            ctx.step(a2, b2, 60_000 + w, out2, closure=1, mlp=mlp_dev); a2, b2 = b2, a2
        f1.record(); f1.synchronize()
        extras["step_with_mlp_closure"] = {"ms_per_step": f0.elapsed_time(f1) / nrep,
                                           "particle_steps_per_s": np_ * nrep / (f0.elapsed_time(f1) * 1e-3)}
        if not args.small:
            del a2, b2, out2
            extras["beyond_l2"] = corroborate(fpcl, torch, workloads, mlp_dev, hbm_peak, min(args.steps, 20))
            extras["paper_surrogate_16_256x4_9"] = paper_surrogate(fpcl, torch, workloads, cfg["tau"])
            extras["c1_couette"] = couette_small(fpcl, torch, workloads)
            extras["c2_closure_microbench"] = closure_microbench(fpcl, torch, workloads, mlp_dev, hbm_peak)
            # BASELINE config 4 asks for the drift after 1,000 steps at every ppc: 0.07 / 0.12 / 0.35 s of GPU time
            extras["c4_ppc_sweep"] = ppc_sweep(fpcl, torch, workloads, 1000, steps_20ppc=1000)

    cpu_baseline = None
    if rank == 0 and not args.no_cpu_baseline:
        # SURVEY 8(d) / BASELINE.md section 3: one thread and all host cores (OpenMP over cells / particles; the sort stays serial)
        v1, done1, dt1, _ = oracle_sample(cfg, settled, args.closure, mlp_host if closure else None, threads=1)
        va, donea, dta, used = oracle_sample(cfg, settled, args.closure, mlp_host if closure else None, threads=0)
        cpu_baseline = {"value": va, "unit": UNIT, "cores": used, "kind": "oracle", "cpu_model": cpu_model(),
                        "value_1_thread": v1,
                        "sample": "%d full fp_step(s) of the same %d-particle ensemble by oracle/ on %d threads (%.1f s), "
                                  "%d on 1 thread (%.1f s)" % (donea, np_, used, dta, done1, dt1)}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": wname, "closure": args.closure, "particles_per_gpu": np_, "cells": ncell,
                           "settle_steps": args.settle, "parallelism": "replicas x%d (independent seeds)" % world,
                           "l2": "working set (two SoA copies + sort scratch = %d MB) exceeds the 126 MB L2; no "
                                 "explicit flush between steps" % ((48 * np_ + 16 * np_) // (1 << 20))},
                "closure_cells_per_s": ncell / (stages["closure"]["ms"] * 1e-3) if stages["closure"]["ms"] > 0 else None,
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "steps": e2e_steps, "api": "fp_step_host (pinned host buffers)"},
                "gpu_launches": int(launches),
                "roofline": roofline, "stages": stages,
                "ms_per_step_with_stage_events": ms_total_staged / args.steps, "cpu_baseline": cpu_baseline,
                "flags_nonzero_cells": int((flags_host != 0).sum())}
        line.update(extras)
        print(json.dumps(line, default=float))
    ctx.close()
    D.shutdown()


if __name__ == "__main__":
    main()
