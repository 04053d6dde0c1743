#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native weighted-NMF hot path.

    python bench.py --gpus N --steps K --warmup W [--impl reference] [--workload stis]

Metric (BASELINE.json): NMF iterations/s at 200 reference frames x 1024^2 px x K=50, fp32.
One "step" is one pass of the whole hot path of SURVEY.md 8(a) over the STIS-shaped
synthetic library: one full NMF iteration (a1-a8: H half-step, W half-step), one
projection iteration of the 32 science frames on the current components (a9) and one
PSF subtraction (a10).  `value` = steps/s summed over all ranks (each rank runs its own
independent replica: weak scaling, no data-path collective).

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "nmf_iterations_per_s@200x1024^2xK50_fp32"
UNIT = "iterations/s"
WORKLOADS = {
    # name: (N, S, K, M)   -- configs[2] of BASELINE.json is the one the metric is quoted on
    "stis": dict(N=200, S=1024, K=50, M=32),
    "stis_small": dict(N=200, S=256, K=50, M=8),     # debugging only
}
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12     # FP32 FFMA: SMs x lanes x 2 x max SM clock


def kernel_sources_sha256():
    """sha256 over the tensor-core kernel sources: profiles/traffic.json records it at capture time, so an ncu byte
    count taken from an older kernel is flagged instead of being reported silently"""
    import hashlib
    h = hashlib.sha256()
    for f in ("nmf_tc.cuh", "nmf_tcfit.cu", "nmf_tcsplit.cu"):
        h.update(open(os.path.join(ROOT, "paper_2309_04623_b200", "csrc", f), "rb").read())
    return h.hexdigest()


def load_traffic(variant):
    """ncu dram bytes per launch of the fit kernel(s) of `variant` from profiles/traffic.json, or (None, why)"""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    except Exception:
        return None, "profiles/traffic.json missing"
    e = t.get(f"variant{variant}")
    if not isinstance(e, dict):
        return None, f"no ncu capture recorded for variant {variant}"
    if e.get("kernel_sha256") != kernel_sources_sha256():
        return None, f"stale: {e.get('source')} was captured from different kernel sources"
    return e.get("dram_bytes_per_launch"), e.get("source")


def flops_per_iter(N, P, K):
    return 12.0 * N * K * P          # six N.K.P contractions


def bytes_per_iter(N, P, K):
    return 8.0 * N * P + 8.0 * K * P  # X, Omega read once; H read + written


# ------------------------------------------------------------------------------
# clocks sampler (nvidia-smi during the timed region)
# ------------------------------------------------------------------------------
class ClockSampler:
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self, t0=None, t1=None):
        import datetime
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = []
        for line in self.f:
            t = [c.strip() for c in line.split(",")]
            if len(t) < 8:
                continue
            try:
                ts = datetime.datetime.strptime(t[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                rows.append((ts, float(t[1]), float(t[2]), float(t[3]), t[4:8]))
            except ValueError:
                continue
        inside = [r for r in rows if t0 is None or (t0 - 0.02 <= r[0] <= t1 + 0.02)]
        window = "timed region"
        if not inside:                      # region shorter than the sampling period: the samples closest to it
            inside = sorted(rows, key=lambda r: abs(r[0] - (t0 or 0)))[:3]
            window = "nearest samples (timed region shorter than the sampling period)"
        for ts, a, b, c, flags in inside:
            sm.append(a); smax.append(b); power.append(c)
            for nm, v in zip(names, flags):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        os.unlink(self.f.name)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None,
                "samples": len(sm), "window": window, "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------
# the CPU oracle legs (cpu_baseline and --impl reference)
# ------------------------------------------------------------------------------
def oracle_step_rate(p, steps: int, warmup: int, budget_s: float):
    """Time the oracle, as it stands, on the workload.  One step = one oracle iteration + one projection
    iteration + subtraction, as in the GPU arm.  The steps run at FULL size when `warmup + steps` of them fit
    `budget_s` (judged from the first, untimed, full-size step); otherwise -- labelled as such -- on a crop: the
    first rows of every frame (all N frames, all K components), the rate scaled by the pixel fraction.
    Returns (full-size steps/s, seconds per timed step as run, threads, description of the sample)."""
    from oracle import nmf_oracle as orc

    def run(Pc, n_warm, n_timed):
        X = np.ascontiguousarray(p.X[:, :Pc]); Om = np.ascontiguousarray(p.Omega[:, :Pc])
        T = np.ascontiguousarray(p.T[:, :Pc]); om = np.ascontiguousarray(p.omega_t[:, :Pc])
        W = p.W0.astype(np.float64); H = np.ascontiguousarray(p.H0[:, :Pc]).astype(np.float64)
        C = p.C0.astype(np.float64)
        dt = []
        for s in range(n_warm + n_timed):
            t0 = time.perf_counter()
            W, H = orc.fit(X, Om, W, H, 1)
            C = orc.project(H, T, om, C, 1)
            orc.subtract(H, T, C, om, None, 0.0)
            dt.append(time.perf_counter() - t0)
        return dt

    warmup = max(warmup, 1)
    first = run(p.P, 1, 0)[0]                       # one full-size step, untimed (first-touch, thread start-up)
    if first * (warmup - 1 + steps) <= budget_s:
        dt = run(p.P, warmup - 1, steps)[warmup - 1:]
        sec = sum(dt) / len(dt)
        sample = (f"{steps} timed full-size steps (+{warmup} warm-up): all {p.P} px of all {p.N} frames, K={p.K}, "
                  f"M={p.M}; {sec:.2f} s per step")
        return 1.0 / sec, sec, orc.num_threads(), sample
    rows = max(1, min(p.S, int(p.S * budget_s / (first * (warmup + steps)))))
    Pc = rows * p.S
    dt = run(Pc, warmup, steps)[warmup:]
    sec = sum(dt) / len(dt)
    sample = (f"CROP (full-size steps would not fit {budget_s:.0f} s: one takes {first:.2f} s): {steps} timed steps "
              f"(+{warmup} warm-up) on the first {rows} image rows ({Pc} of {p.P} px) of all {p.N} frames, K={p.K}, "
              f"{sec:.3f} s per crop step; rate scaled by the pixel fraction")
    return (1.0 / sec) * (Pc / p.P), sec, orc.num_threads(), sample


def run_reference(args, rank):
    """--impl reference: the fp64 oracle on the host cores (rank 0 only)."""
    if rank != 0:
        return
    from paper_2309_04623_b200 import inputs
    wl = WORKLOADS[args.workload]
    p = inputs.make_stis(N=wl["N"], S=wl["S"], K=wl["K"], M=wl["M"])
    rate, sec, cores, sample = oracle_step_rate(p, args.steps, max(args.warmup, 1), args.cpu_budget)
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / rate, "measured_s_per_step": sec,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "gpu_launches": 0,
            "config": {"workload": f"STIS-shaped N={p.N} {p.S}x{p.S}px K={p.K} M={p.M} (BASELINE.json configs[2])",
                       "step": "1 NMF iteration + 1 projection iteration + subtraction", "sample": sample},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ------------------------------------------------------------------------------
# the GPU arm
# ------------------------------------------------------------------------------
def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2309_04623_b200 import inputs, nmf, sharding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    # nvidia-smi needs a few hundred ms for its first sample: start it now, keep only the samples whose time stamp
    # falls inside the timed region
    sampler = ClockSampler(local_rank) if rank == 0 else None
    wl = WORKLOADS[args.workload]
    # every rank fits its own replica (per-rank seed): independent problems, no collective
    p = inputs.make_stis(N=wl["N"], S=wl["S"], K=wl["K"], M=wl["M"], seed=sharding.replica_seed(3003, rank))
    N, P, K, M = p.N, p.P, p.K, p.M
    plan = nmf.Plan(N, P, K, max_targets=M, variant=args.variant)
    pin = lambda a: torch.from_numpy(a).pin_memory()
    hX, hOm, hT, hom = pin(p.X), pin(p.Omega), pin(p.T), pin(p.omega_t)
    X, Om, T, om = hX.cuda(non_blocking=True), hOm.cuda(non_blocking=True), hT.cuda(non_blocking=True), hom.cuda(non_blocking=True)
    W, H, C = torch.from_numpy(p.W0).cuda(), torch.from_numpy(p.H0).cuda(), torch.from_numpy(p.C0).cuda()
    out = torch.empty_like(T)
    torch.cuda.synchronize()

    def step():
        plan.fit(X, Om, W, H, 1)
        plan.project(H, T, om, C, 1)
        plan.subtract(H, T, C, om, None, 0.0, out)

    for _ in range(args.warmup):
        step()
    ev = lambda: torch.cuda.Event(enable_timing=True)
    fit_ev = [(ev(), ev()) for _ in range(args.steps)]
    e0, e1 = ev(), ev()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    l0 = plan.launch_count
    t_wall0 = time.time()
    e0.record()
    for s in range(args.steps):
        fit_ev[s][0].record()
        plan.fit(X, Om, W, H, 1)
        fit_ev[s][1].record()
        plan.project(H, T, om, C, 1)
        plan.subtract(H, T, C, om, None, 0.0, out)
    e1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop(t_wall0, time.time()) if sampler else None
    launches = plan.launch_count - l0
    ms_total = e0.elapsed_time(e1)
    fit_ms = [a.elapsed_time(b) for a, b in fit_ev]
    ms_max = sharding.max_over_ranks(ms_total, "cuda")
    assert torch.isfinite(W).all() and torch.isfinite(H).all()

    # ---- end-to-end through the C-ABI with host buffers (copies inside the timed region) ----
    hW, hH, hC = pin(p.W0.copy()), pin(p.H0.copy()), pin(p.C0.copy())
    hout = torch.empty(M, P).pin_memory()
    e2e_iters = args.steps

    def e2e_call():
        plan.fit_host(hX, hOm, hW, hH, e2e_iters)
        Hd = torch.empty(K, P, device="cuda"); Hd.copy_(hH, non_blocking=True)
        plan.project_subtract_host(Hd, hT, hom, hC, hout, e2e_iters)

    plan.use_own_staging(M)                       # the staging of the *_host calls is a torch tensor of this process
    hW.copy_(torch.from_numpy(p.W0)); hH.copy_(torch.from_numpy(p.H0))
    e2e_call()                                    # warm-up
    hW.copy_(torch.from_numpy(p.W0)); hH.copy_(torch.from_numpy(p.H0)); hC.copy_(torch.from_numpy(p.C0))
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    e2e_call()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s = sharding.max_over_ranks(e2e_s, "cuda")
    h2d = 4.0 * (2 * N * P + N * K + K * P) + 4.0 * (K * P + 2 * M * P + M * K)
    d2h = 4.0 * (N * K + K * P) + 4.0 * (M * K + M * P)

    if rank != 0:
        return
    value = world * args.steps / (ms_max * 1e-3)
    fit_ms_avg = sum(fit_ms) / len(fit_ms)
    F = flops_per_iter(N, P, K)
    achieved = F / (fit_ms_avg * 1e-3) / 1e12
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    traffic, traffic_note = load_traffic(plan.variant)
    cpu = None
    if not args.no_cpu_baseline:
        rate, sec, cores, sample = oracle_step_rate(p, 2, 1, 60.0)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    roof_common = {"traffic": traffic, "algorithmic_flops_per_launch": F,
                   "algorithmic_bytes_per_launch": bytes_per_iter(N, P, K),
                   "hbm_time_floor_ms": bytes_per_iter(N, P, K) / (hbm_peak * 1e9) * 1e3,
                   "hbm_peak_gbs_measured": hbm_peak,
                   "achieved_gbs_algorithmic": bytes_per_iter(N, P, K) / (fit_ms_avg * 1e-3) / 1e9}
    if plan.variant in (3, 4):
        # BF16x3: every FP32 product is six BF16 tensor-core products, so the pipe peak for
        # the ALGORITHMIC 12NKP flops is the measured dense BF16 rate / 6.  The BURST figure is the denominator: the
        # timed region is tens of milliseconds at full SM clock, not the seconds-long power-capped regime of the
        # sustained figure (kept as frac_of_sustained_peak).
        bf16 = peaks.get("bf16_tflops", 1590.0)
        bf16_s = peaks.get("bf16_tflops_sustained", 1400.0)
        tpeak = bf16 / 6.0
        roofline = {"bound": "tensor", "achieved": achieved, "peak": tpeak, "unit": "TFLOP/s", "frac": achieved / tpeak,
                    "kernel": ("fit iteration (k_tc_iter: tcgen05 BF16x3 fused tile kernel, + fixed-order reduce/W update)"
                               if plan.variant == 3 else
                               "fit iteration (k_tc_h + k_tc_w: tcgen05 BF16x3 half-step kernels, + fixed-order reduce/W update)"),
                    "peak_source": (f"MEASURED_PEAKS.json bf16_tflops (burst, {bf16}) / 6 piece products per FP32 product"
                                    if peaks else "fallback 1590 TF/s burst bf16 / 6 (B200_PROFILING.md)"),
                    "tensor_time_floor_ms": F / (tpeak * 1e12) * 1e3,
                    "frac_of_sustained_peak": achieved / (bf16_s / 6.0),
                    "frac_of_ffma_roofline": achieved / ALU_PEAK_TFLOPS, "traffic_note": traffic_note, **roof_common}
    elif plan.variant == 5:
        # K <= 8: 12NKP flops are a fraction of the FP32 pipe; the kernel streams X and Omega once: HBM-bound
        gbs = bytes_per_iter(N, P, K) / (fit_ms_avg * 1e-3) / 1e9
        roofline = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                    "kernel": "fit iteration (k_stream: streaming FP32 kernel, K <= 8, + fixed-order reduce/W update)",
                    "peak_source": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback (B200_PROFILING.md)",
                    "traffic_note": traffic_note, **roof_common}
    else:
        roofline = {"bound": "alu", "achieved": achieved, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s",
                    "frac": achieved / ALU_PEAK_TFLOPS,
                    "kernel": "fit iteration (fused tile kernel + fixed-order reduce/W update)" if plan.variant == 2
                              else "fit iteration (H half-step + W half-step partial + reduce kernels)",
                    "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (B200_PROFILING.md unit counts/clocks)",
                    **roof_common}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"STIS-shaped N={N} {p.S}x{p.S}px K={K} M={M} (BASELINE.json configs[2])",
                   "step": "1 NMF iteration (a1-a8) + 1 projection iteration of M frames (a9) + subtraction (a10)",
                   "fit_variant": {1: "generic two-kernel", 2: "fused per-pixel-tile FFMA",
                                   3: "fused per-pixel-tile tcgen05 BF16x3",
                                   4: "split tcgen05 BF16x3 (H half-step kernel + W half-step kernel)",
                                   5: "streaming FP32 kernel (K <= 8)",
                                   6: "resident kernel (whole fit in one cooperative launch)"}[plan.variant],
                   "l2": "inputs (X+Omega 1.6 GB per step) are larger than the 126 MB L2; no explicit flush",
                   "parallelism": f"{world} independent replica(s), no collective"},
        "fit_ms_per_iter": fit_ms_avg,
        "fit_iterations_per_s": 1e3 / fit_ms_avg,
        "roofline": roofline,
        "e2e": {"value": world * e2e_iters / e2e_s, "unit": UNIT,
                "h2d_bytes_per_step": h2d / e2e_iters, "d2h_bytes_per_step": d2h / e2e_iters,
                "call": f"nmf_fit_host(iters={e2e_iters}) + nmf_project_subtract_host(iters={e2e_iters}) with pinned "
                        f"host buffers; all H2D/D2H copies inside the timed region, amortised over {e2e_iters} iterations"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line))


def run_configs(args):
    """--configs: fit-iteration rate of every BASELINE.json config (CUDA events around nmf_fit / nmf_fit_batched
    on random data of each config's shape; throughput does not depend on the values).  A secondary table for
    DESIGN.md; the driver's contract line is the default mode."""
    import torch
    from paper_2309_04623_b200 import nmf
    torch.cuda.set_device(0)
    rows = [("tiny", 1, 16, 64 * 64, 5), ("MIRI-shaped", 1, 96, 256 * 256, 30), ("STIS-shaped", 1, 200, 1024 * 1024, 50)]
    rows += [(f"sweep K={K}", 1, 200, 1024 * 1024, K) for K in (1, 5, 10, 20, 50, 100)]
    rows += [("survey batch (64 problems)", 64, 128, 256 * 256, 20)]
    out = {}
    for name, B, N, P, K in rows:
        plan = nmf.Plan(N, P, K, batch=B, variant=args.variant)
        shp = (lambda *d: (B, *d)) if B > 1 else (lambda *d: d)
        X = torch.rand(shp(N, P), device="cuda") * 10
        Om = torch.rand(shp(N, P), device="cuda"); Om = Om * (Om > 0.1)
        W = torch.rand(shp(N, K), device="cuda") + 0.1
        H = torch.rand(shp(K, P), device="cuda") + 0.1
        fit = plan.fit_batched if B > 1 else plan.fit
        iters = max(3, min(200, int(2e11 / (12.0 * B * N * K * P))))
        try:
            fit(X, Om, W, H, 3)
        except nmf.NMFError as e:                        # a forced family that does not cover this shape
            print(f"[configs] {name}: variant {args.variant} unsupported ({e})", file=sys.stderr, flush=True)
            out[name] = {"variant": args.variant, "unsupported": True}
            del plan, X, Om, W, H
            torch.cuda.empty_cache()
            continue
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(); fit(X, Om, W, H, iters); e1.record(); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / iters
        F, Bt = flops_per_iter(N, P, K) * B, bytes_per_iter(N, P, K) * B
        print(f"[configs] {name}: variant {plan.variant} {ms:.4f} ms/iteration", file=sys.stderr, flush=True)
        out[name] = {"variant": plan.variant, "ms_per_iteration": ms, "iterations_per_s": 1e3 / ms,
                     "algorithmic_tflops": F / ms / 1e9, "algorithmic_gbs": Bt / ms / 1e6}
        del plan, X, Om, W, H
        torch.cuda.empty_cache()
    print(json.dumps({"configs": out}))


def run_trace(args):
    """--trace: timeline of one persistent CTA of the split tensor-core kernels at the metric's shape.  Builds the
    library with -DNMF_TC_TRACE (paper_2309_04623_b200/build/libnmf_trace.so; the product library is untouched), runs
    one fit iteration (k_tc_h, k_tc_w) on random data of the workload's shape and prints, as markdown, where the
    element-wise groups and the MMA issuer of CTA (0, 0, 0) spent their cycles (steady-state tiles only)."""
    import ctypes
    import torch
    from paper_2309_04623_b200 import build as nmf_build, nmf
    nmf.LIB_PATH = nmf_build.build_trace()
    torch.cuda.set_device(0)
    wl = WORKLOADS[args.workload]
    N, P, K = wl["N"], wl["S"] * wl["S"], wl["K"]
    plan = nmf.Plan(N, P, K, variant=4)
    X = torch.rand(N, P, device="cuda") * 10
    Om = torch.rand(N, P, device="cuda"); Om = Om * (Om > 0.1)
    W = torch.rand(N, K, device="cuda") + 0.1
    H = torch.rand(K, P, device="cuda") + 0.1
    L = nmf.lib()
    NW, LEN = 18, 2048
    counts = (ctypes.c_uint * (2 * NW))()
    events = (ctypes.c_ulonglong * (2 * NW * LEN))()
    L.nmf_debug_trace.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
    plan.fit(X, Om, W, H, 2); torch.cuda.synchronize()
    L.nmf_debug_trace(counts, events, 1)
    plan.fit(X, Om, W, H, 1); torch.cuda.synchronize()
    L.nmf_debug_trace(counts, events, 1)
    names = {1: "slot landed", 2: "S ready", 3: "S loaded", 4: "piece columns free", 5: "chunk handed over",
             6: "H pieces begin", 7: "H pieces done", 8: "update begin", 9: "update done", 10: "previous tile's MMAs complete",
             11: "H slot landed", 16: "chunk ready", 17: "chunk MMAs issued", 18: "S series issued", 19: "H pieces ready",
             24: "ring slot acquired"}
    if args.trace_raw:                                   # every event of every warp: kernel, warp, event, argument, clock64
        with open(args.trace_raw, "w") as f:
            f.write("kernel,warp,event,arg,clock\n")
            for ki, kern in enumerate(("k_tc_h", "k_tc_w")):
                for w in range(NW):
                    for i in range(min(counts[ki * NW + w], LEN)):
                        e = events[(ki * NW + w) * LEN + i]
                        f.write(f"{kern},{w},{names.get((e >> 56) & 0xff, (e >> 56) & 0xff)},{(e >> 48) & 0xff},{e & 0xffffffffffff}\n")
    print(f"# Timeline of CTA (0,0,0), split tensor-core kernels, N={N} P={P} K={K} (cycles of clock64)\n")
    print("Command: `python bench.py --trace` (builds build/libnmf_trace.so with -DNMF_TC_TRACE; one fit iteration on random data)\n")
    for ki, kern in enumerate(("k_tc_h", "k_tc_w")):
        print(f"## {kern}\n")
        per_warp = {}
        for w in range(NW):
            ev = [events[(ki * NW + w) * LEN + i] for i in range(min(counts[ki * NW + w], LEN))]
            ev = [((e >> 56) & 0xff, (e >> 48) & 0xff, e & 0xffffffffffff) for e in ev]
            if ev:
                per_warp[w] = ev
        if not per_warp:
            print("(no events)\n"); continue
        t_all = [t for ev in per_warp.values() for _, _, t in ev]
        span = max(t_all) - min(t_all)
        print(f"events recorded over {span} cycles (log capacity {LEN} events per warp)\n")
        print("| warp | role | mean cycles between consecutive events (from -> to: mean x count) |")
        print("|---|---|---|")
        for w, ev in sorted(per_warp.items()):
            gaps = {}
            for (e0, a0, t0), (e1, a1, t1) in zip(ev[len(ev) // 4:], ev[len(ev) // 4 + 1:]):     # skip the start-up quarter
                gaps.setdefault((e0, e1), []).append(t1 - t0)
            role = ("TMA producer" if any(e >= 24 for e, _, _ in ev) else "MMA issuer" if any(e >= 16 for e, _, _ in ev)
                    else f"element-wise, group {w // 4}, quadrant {w % 4}")
            txt = "; ".join(f"{names.get(a, a)} -> {names.get(b, b)}: {sum(v) / len(v):.0f} x {len(v)}"
                            for (a, b), v in sorted(gaps.items(), key=lambda kv: -sum(kv[1]))[:8])
            if w % 4 == 0 or not role.startswith("element"):
                print(f"| {w} | {role} | {txt} |")
        print()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="stis", choices=sorted(WORKLOADS))
    ap.add_argument("--variant", type=int, default=0, help="0 auto, 1 generic, 2 fused FFMA, 3 fused tensor core, 4 split tensor core, 5 streaming FP32 (K <= 8), 6 resident (small problems)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=420.0,
                    help="--impl reference: seconds of oracle steps allowed at full size before falling back to a crop")
    ap.add_argument("--configs", action="store_true", help="print the fit-iteration rate of every config and exit")
    ap.add_argument("--trace", action="store_true", help="print the tile timeline of the split tensor-core kernels (markdown) and exit")
    ap.add_argument("--trace-raw", default="", help="with --trace: also write every recorded event to this CSV file")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.trace:
        if rank == 0:
            run_trace(args)
    elif args.configs:
        if rank == 0:
            run_configs(args)
    elif args.impl == "reference":
        run_reference(args, rank)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
