#!/usr/bin/env python
"""bench.py -- one JSON line for the CROWN hot path on B200 (contract: DESIGN.md sec. "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl b200|reference]

A "step" is one pass of the whole hot path (IBP -> CROWN intermediate bounds for every ReLU -> (alpha-)CROWN final
bound -> concretisation -> verdict) over one batch of synthetic input.
Headline workload = BASELINE.json configs[2] (cfg3): the largest single-GPU configuration, wide MLP
4096-16384x3-10, 16 properties, 9 margin specs, full CROWN row-chunked under a 64 GiB workspace cap (BASELINE.md
sec. 3 puts the tensor-roofline target on cfg3 / cfg4).  The same JSON line carries a `per_config` object with the
other four configs (fewer steps for the long ones).  Inputs are seeded and synthetic (workloads.py); they stand in
for the paper's VNN-COMP / wide-MLP workloads, which are not reproduced.

value  : properties/s, device-timed (CUDA events on the launching stream), inputs resident in HBM.
e2e    : same metric through crown_run_host: pinned HOST buffers, H2D of x_lo/x_hi/C/alpha and D2H of
         lb/ub/verified inside the timed region.
Multi-GPU (torchrun): properties are independent, every rank runs its own batch (weak scaling), no
data-path collective; time = max over ranks.
--impl reference: the float64 CPU oracle (oracle/) as it stands, on a bounded sample per step.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

METRIC, UNIT = "properties_per_sec", "properties/s"
TF32_OVER_BF16 = 1.1 / 2.25          # nominal dense ratio (B200_PROFILING.md table); used only if TF32 is not measured
ALL_CFGS = ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"]


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=ALL_CFGS)
    ap.add_argument("--no-per-config", action="store_true", help="only the --workload config (no per_config block)")
    ap.add_argument("--scale", type=int, default=1, help="width divisor (debug only; 1 = the named config)")
    ap.add_argument("--batch", type=int, default=0, help="override B (debug only)")
    ap.add_argument("--mem-cap-gb", type=float, default=0.0)
    ap.add_argument("--stream-weights", action="store_true",
                    help="layers with >= 2^28 weights are streamed from pinned host memory (a7), not resident")
    ap.add_argument("--no-epi-fusion", action="store_true", help="run the relaxation as its own kernel (debug)")
    ap.add_argument("--k-drain", type=int, default=0, help="3xTF32 drain chunk (debug; 0 = library default)")
    ap.add_argument("--no-graph", action="store_true", help="do not replay crown_run from a CUDA graph (debug)")
    ap.add_argument("--no-conv-tc", action="store_true", help="BoundConv backward on the CUDA-core kernel everywhere (debug)")
    ap.add_argument("--alpha-iters", type=int, default=10,
                    help="alpha-mode configs: also time this many projected ascent steps on alpha (NEXT-1; 0 = skip)")
    ap.add_argument("--bab-domains", type=int, default=4096,
                    help="cfg2: also time the joint alpha/beta ascent (NEXT-2) on this many BaB sub-domains (0 = skip)")
    ap.add_argument("--shard-rows", action="store_true",
                    help="NEXT-4 (opt-in, torchrun): all ranks work on the SAME batch; the identity rows of every intermediate "
                         "pass are sharded across ranks, one AllGather of (l_k, u_k) per layer (strong scaling)")
    ap.add_argument("--no-conv-crown", action="store_true", help="cfg5: skip the CROWN-intermediate-bounds leg (NEXT-3)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--device-steps-only", action="store_true",
                    help="profiling aid (ncu): only the warm-up and the timed device steps of --workload; no TF32 peak "
                         "measurement, end-to-end leg, per-class timing leg, alpha leg, CPU baseline or per_config")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm": d["hbm_gbs"], "bf16": d["bf16_tflops"], "bf16_sustained": d["bf16_tflops_sustained"],
                "src": "measured"}
    return {"hbm": 6650.0, "bf16": 1590.0, "bf16_sustained": 1400.0, "src": "fallback"}


def kernel_source_sha1(files):
    """sha1 over the CUDA sources a kernel is built from: a committed ncu traffic figure is only quoted while they are unchanged."""
    h = hashlib.sha1()
    d = os.path.join(ROOT, "paper_2606_09377_b200", "csrc")
    for f in sorted(files):
        with open(os.path.join(d, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def profiled_traffic(cfgname, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed ncu --set full capture of
    this workload (profiles/traffic.json: {"cfgN:kernel": {dram_bytes_per_launch, src_files, src_sha1, profile}}), or None
    when there is none for the current sources of that kernel."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        tab = json.load(f)
    e = tab.get(f"{cfgname}:{kernel}")
    if not e or e.get("src_sha1") != kernel_source_sha1(e.get("src_files", [])):
        return None
    return {"dram_bytes_per_launch": e["dram_bytes_per_launch"], "launch": e.get("launch"), "profile": e.get("profile")}


def workload_desc(wl, cfgname):
    return {"workload": f"{cfgname}:{wl.name}", "B": int(wl.B), "S": int(wl.S),
            "eps_set": sorted({round(float(e), 6) for e in wl.eps}), "properties_per_step": int(wl.B),
            "intermediate": wl.intermediate, "alpha": wl.alpha is not None}


def make_workload(cfgname, args):
    cfg = int(cfgname[3:])
    return W.stack_eps(W.make(cfg, scale=args.scale, B=args.batch or None))


# ------------------------------------------------------------------------------------------------
# oracle legs (cpu_baseline and --impl reference): the ONLY places bench.py executes oracle/
# ------------------------------------------------------------------------------------------------
def cpu_info():
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    blas, thr = "unknown", os.cpu_count() or 1
    try:
        from threadpoolctl import threadpool_info
        info = threadpool_info()
        if info:
            blas = ", ".join(sorted({f"{p.get('internal_api')} {p.get('version')}" for p in info}))
            thr = max(p.get("num_threads", 1) for p in info)
    except Exception:
        pass
    return model, blas, thr


def oracle_props(wl, budget_s, max_props=None):
    """Runs the float64 oracle, as it stands, on whole properties (eps groups round robin) until budget_s is spent
    (at least one property).  Returns (properties done, seconds)."""
    from oracle import crown_oracle as O
    lo, hi = wl.box()
    done, t0 = 0, time.perf_counter()
    k = max(1, len({float(e) for e in wl.eps}))
    per = max(1, wl.B // k)
    for p in sorted(range(wl.B), key=lambda q: (q % per, q // per)):
        al = None if wl.alpha is None else [a[p] for a in wl.alpha]
        O.run_property(wl.net, lo[p], hi[p], wl.C[p], al, wl.intermediate)
        done += 1
        if time.perf_counter() - t0 >= budget_s or (max_props and done >= max_props):
            break
    return done, time.perf_counter() - t0


def oracle_rows_time(wl, frac, p=0):
    """Seconds the oracle needs for the intermediate bounds (O4) of property p when only the first ceil(frac * n_k)
    identity rows of every CROWN pass are propagated (rows are independent linear bounds)."""
    from oracle import crown_oracle as O
    lo, hi = wl.box()
    rows = {i: np.arange(max(1, int(np.ceil(frac * wl.net.nodes[i].size)))) for i in wl.net.relu_ids()}
    t0 = time.perf_counter()
    O.crown_bounds(wl.net, lo[p], hi[p], wl.intermediate, rows=rows)
    return time.perf_counter() - t0


def oracle_final_time(wl, p=0):
    """Seconds of the oracle's final pass (O5) for property p; intermediate bounds = IBP (the arithmetic and its cost
    do not depend on their values)."""
    from oracle import crown_oracle as O
    lo, hi = wl.box()
    ib = O.ibp(wl.net, lo[p], hi[p])
    pre = {i: (ib[wl.net.nodes[i].in0][0].reshape(-1), ib[wl.net.nodes[i].in0][1].reshape(-1)) for i in wl.net.relu_ids()}
    t0 = time.perf_counter()
    O.final_bounds(wl.net, lo[p], hi[p], wl.C[p], pre, None, None)
    return time.perf_counter() - t0


LARGE = ("cfg3", "cfg4")
F1, F2 = 1.0 / 64, 1.0 / 16            # row fractions of the two sampled runs (cfg3: 256 and 1024 of 16384 rows)


def oracle_baseline(wl, cfgname, budget_s):
    """cpu_baseline object: whole properties for cfg1/2/5; for cfg3/cfg4 one property is timed on two row samples
    (F1 and F2 of every identity pass) and extrapolated linearly in the row count -- stated as scaled."""
    model, blas, thr = cpu_info()
    base = {"unit": UNIT, "cores": thr, "kind": "oracle", "cpu_model": model, "blas": blas}
    if cfgname not in LARGE:
        n, secs = oracle_props(wl, budget_s)
        base.update(value=n / secs, sample=f"first {n} of {wl.B} properties (eps round robin), {secs:.1f} s, float64 numpy")
        try:
            from threadpoolctl import threadpool_limits
            with threadpool_limits(limits=1):
                n1, s1 = oracle_props(wl, min(budget_s, 6.0))
            base["single_thread_value"] = n1 / s1
        except Exception:
            base["single_thread_value"] = None
        return base
    t1 = oracle_rows_time(wl, F1)
    t2 = oracle_rows_time(wl, F2)
    tf = oracle_final_time(wl)
    slope = max(t2 - t1, 0.0) / (F2 - F1)
    t_full = t2 + slope * (1.0 - F2) + tf
    base.update(value=1.0 / t_full, single_thread_value=None,
                sample=f"1 property, identity rows sampled at {F1:.5f} ({t1:.1f} s) and {F2:.5f} ({t2:.1f} s) of every "
                       f"CROWN pass + final pass ({tf:.1f} s), extrapolated linearly to all rows: {t_full:.0f} s per "
                       "property (SCALED, not run in full), float64 numpy")
    return base


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(args.workload, args)
    model, blas, thr = cpu_info()
    if args.workload in LARGE:
        t1 = oracle_rows_time(wl, F1)               # calibration of the fixed part, once (the warm-up step)
        tf = oracle_final_time(wl)
        tot_t = 0.0
        for _ in range(args.steps):
            t2 = oracle_rows_time(wl, F2)
            slope = max(t2 - t1, 0.0) / (F2 - F1)
            tot_t += t2 + slope * (1.0 - F2) + tf
        v = args.steps / tot_t
        ms = 1e3 * tot_t / args.steps
        sample = (f"per step: 1 property with {F2:.5f} of the identity rows of every CROWN pass, extrapolated linearly "
                  f"to all rows with the fixed part calibrated once at {F1:.5f} (SCALED), float64 numpy")
    else:
        n1, t1 = oracle_props(wl, 0.0, max_props=1)
        per_step = max(1, min(wl.B, int(5.0 / max(t1 / n1, 1e-6))))
        for _ in range(min(args.warmup, 1)):
            oracle_props(wl, 1e9, max_props=per_step)
        tot_n, tot_t = 0, 0.0
        for _ in range(args.steps):
            n, t = oracle_props(wl, 1e9, max_props=per_step)
            tot_n += n
            tot_t += t
        v = tot_n / tot_t
        ms = 1e3 * tot_t / args.steps
        sample = f"{per_step} of {wl.B} properties per step (first ones, eps round robin), float64 numpy"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_desc(wl, args.workload),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": sample,
                         "cpu_model": model, "blas": blas},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------
# clocks during the timed region (NVML; the recipe's clocks line)
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz, self.ok = [], set(), None, False
        self._stop = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "sw_power_cap": 0x4, "hw_power_brake_slowdown": 0x80}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.05)

    def start(self):
        if self.ok:
            self.t.start()

    def stop(self):
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable"]}
        self._stop.set()
        self.t.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}


def measure_tf32_peak(dev):
    """Dense TF32 tensor throughput of this box, measured the way MEASURED_PEAKS.json measures bf16: torch.matmul
    (cuBLAS) on 8192^3 fp32 operands with TF32 allowed, best of 10 (burst) and back to back for ~2 s (sustained).
    A measuring stick only: no library GEMM is on the hot path."""
    import torch
    old = torch.backends.cuda.matmul.allow_tf32
    torch.backends.cuda.matmul.allow_tf32 = True
    try:
        n = 8192
        a = torch.randn(n, n, device=dev)
        b = torch.randn(n, n, device=dev)
        for _ in range(3):
            a @ b
        torch.cuda.synchronize()
        best = 1e9
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); a @ b; e1.record(); e1.synchronize()
            best = min(best, e0.elapsed_time(e1))
        reps = max(10, int(2000.0 / best))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            a @ b
        e1.record(); e1.synchronize()
        sus = e0.elapsed_time(e1) / reps
        fl = 2.0 * n ** 3
        return {"burst": fl / (best * 1e-3) / 1e12, "sustained": fl / (sus * 1e-3) / 1e12}
    finally:
        torch.backends.cuda.matmul.allow_tf32 = old


# ------------------------------------------------------------------------------------------------
# the CUDA arm: one configuration
# ------------------------------------------------------------------------------------------------
def measure_config(cfgname, args, steps, warmup, dev, local, world, tf32_peak, with_cpu):
    import gc
    import torch
    import torch.distributed as dist
    from paper_2606_09377_b200 import CrownContext, multi

    cfg = int(cfgname[3:])
    wl = make_workload(cfgname, args)
    lo, hi = wl.box()
    B, S = wl.B, wl.S
    cap = int(args.mem_cap_gb * (1 << 30))
    if cap == 0 and cfg in (3, 4):
        cap = 64 << 30
    free0, _ = torch.cuda.mem_get_info(dev)
    ctx = CrownContext(wl.net, B, S, device=f"cuda:{local}", mem_cap_bytes=cap,
                       stream_weights=int(args.stream_weights), disable_epi_fusion=int(args.no_epi_fusion),
                       disable_graph=int(args.no_graph), disable_conv_tc=int(args.no_conv_tc), k_drain=args.k_drain)
    inter = 1 if wl.intermediate == "ibp" else 0

    # ---- inputs resident in HBM -------------------------------------------------------------------
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    xlo, xhi, Cd = t(lo), t(hi), t(wl.C)
    alpha = None if wl.alpha is None else {i: t(a) for i, a in zip(ctx.relu_ids, wl.alpha)}
    io = ctx.alloc_io(B, S)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def step_device():
        if args.shard_rows:
            r = multi.crown_run_row_sharded(ctx, xlo, xhi, Cd, alpha, int(os.environ.get("RANK", "0")), world)
            io["lb"], io["ub"], io["verified"] = r["lb"], r["ub"], r["verified"]
            return
        ctx.run_device(xlo, xhi, Cd, alpha, inter, io)

    # ---- pinned host buffers for the end-to-end leg ---------------------------------------------------
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_xlo, h_xhi, h_C = pin(lo), pin(hi), pin(wl.C)
    h_alpha = None if wl.alpha is None else [pin(a) for a in wl.alpha]
    h_lb = torch.empty(B, S).pin_memory()
    h_ub = torch.empty(B, S).pin_memory()
    h_ver = torch.empty(B, dtype=torch.uint8).pin_memory()
    h2d = 2 * B * ctx.n0 * 4 + h_C.numel() * 4 + (sum(a.numel() for a in h_alpha) * 4 if h_alpha else 0)
    d2h = 2 * B * S * 4 + B

    def step_host():
        ctx.run_host(h_xlo.numpy(), h_xhi.numpy(), h_C.numpy(),
                     None if h_alpha is None else [a.numpy() for a in h_alpha], wl.intermediate,
                     h_lb.numpy(), h_ub.numpy(), h_ver.numpy())

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, n, w, host_clock=False):
        for _ in range(w):
            fn()
        barrier()
        ms = []
        for _ in range(n):
            flush.fill_(1)                       # L2 flush between timed iterations (outside the event pair)
            torch.cuda.synchronize()
            if host_clock:
                t0 = time.perf_counter()
                fn()
                torch.cuda.synchronize()
                ms.append(1e3 * (time.perf_counter() - t0))
            else:
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                fn()
                b.record()
                b.synchronize()
                ms.append(a.elapsed_time(b))
        barrier()
        return multi.max_over_ranks(sum(ms)) / n       # the job is as slow as its slowest replica

    clk = ClockSampler(local)
    k0 = ctx.launch_count()
    step_device()
    torch.cuda.synchronize()
    launches_per_step = ctx.launch_count() - k0
    free1, _ = torch.cuda.mem_get_info(dev)
    f0 = ctx.gemm_flops()
    clk.start()
    ms_step = timed(step_device, steps, max(warmup - 1, 0))
    clocks = clk.stop()
    nrun = steps + max(warmup - 1, 0)
    flops_step = (ctx.gemm_flops() - f0) / nrun
    w_h2d_step = ctx.h2d_bytes() / (nrun + 1)
    verified = int(io["verified"].sum().item())
    # long steps: the end-to-end and the instrumented legs run fewer steps (they re-measure the same kernels)
    n_aux = steps if ms_step < 200.0 else max(2, min(steps, int(15000.0 / ms_step)))
    if args.device_steps_only or args.shard_rows:
        out = {"value": (B if args.shard_rows else world * B) / (ms_step * 1e-3), "unit": UNIT, "steps": steps, "ms_per_step": ms_step,
               "config": workload_desc(wl, cfgname), "gpu_launches_per_step": int(launches_per_step), "clocks": clocks,
               "aw_flops_per_step": flops_step}
        ctx.close()
        return out
    ms_e2e = timed(step_host, n_aux, 1 if ms_step >= 200.0 else max(warmup, 1), host_clock=True)

    # ---- per-kernel-class device times (CUDA events around every launch; graph replay is off for this leg) ----------
    ctx.timing(True)
    for _ in range(n_aux):
        flush.fill_(1)
        step_device()
    torch.cuda.synchronize()
    classes = ctx.timing_read()
    ctx.timing(False)
    tot_class_ms = sum(c["ms"] for c in classes.values()) or 1.0
    dom = max(classes, key=lambda k: classes[k]["ms"])
    pk = peaks()
    long_step = ms_step > 1000.0
    shares = {k: round(c["ms"] / tot_class_ms, 4) for k, c in classes.items() if c["launches"]}
    # per kernel class: launches per step, mean device time, achieved ALGORITHMIC GB/s and TFLOP/s (bytes / flops are
    # the library's own per-launch algorithmic counts; rows shared by all branches / properties at
    # the start of a pass are counted once)
    per_class = {k: {"launches_per_step": c["launches"] / n_aux, "ms_per_step": c["ms"] / n_aux,
                     "gbs": (c["bytes"] / (c["ms"] * 1e-3) / 1e9) if c["ms"] > 0 and c["bytes"] > 0 else None,
                     "tflops": (c["flops"] / (c["ms"] * 1e-3) / 1e12) if c["ms"] > 0 and c["flops"] > 0 else None}
                 for k, c in classes.items() if c["launches"]}
    d = classes[dom]
    avg_ms = d["ms"] / max(d["launches"], 1)
    # fp32-equivalent tensor peak = TF32 dense / 3 (three TF32 MMAs per useful product).  Two estimates of the TF32 dense
    # rate: measured in this run (cuBLAS TF32 8192^3) and the driver-measured bf16 rate x the nominal TF32/bf16 ratio;
    # the LARGER one is the denominator (cuBLAS TF32 measured below half of its bf16 rate on this pool)
    which = "sustained" if long_step else "burst"
    bf16 = pk["bf16_sustained"] if long_step else pk["bf16"]
    tf32_nom = bf16 * TF32_OVER_BF16
    tf32_meas = tf32_peak[which] if tf32_peak else 0.0
    tc_peak = max(tf32_meas, tf32_nom) / 3.0
    tc_src = (f"max(TF32 dense measured in this run {tf32_meas:.0f}, {pk['src']} bf16 {bf16:.0f} x nominal ratio "
              f"{TF32_OVER_BF16:.3f} = {tf32_nom:.0f}) TFLOP/s {which} / 3")
    g = classes["gemm_tc"]
    aw_tflops = (g["flops"] / (g["ms"] * 1e-3) / 1e12) if g["ms"] > 0 else None
    if dom == "gemm_tc":
        ach = d["flops"] / (d["ms"] * 1e-3) / 1e12
        roof = {"kernel": "gemm2_tf32x3_kernel", "bound": "tensor", "achieved": ach, "peak": tc_peak, "unit": "TFLOP/s",
                "frac": ach / tc_peak, "traffic": profiled_traffic(cfgname, "gemm2_tf32x3_kernel"), "peak_source": tc_src}
    elif dom == "conv":
        # CUDA-core FFMA peak: SMs x 128 lanes x 2 flop x SM clock under load
        sm_clk = (clocks.get("sm_mhz") or 1965.0) * 1e6
        peak = 148 * 128 * 2 * sm_clk / 1e12
        ach = d["flops"] / (d["ms"] * 1e-3) / 1e12
        roof = {"kernel": "conv backward / conv IBP", "bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                "frac": ach / peak, "traffic": profiled_traffic(cfgname, "conv"),
                "peak_source": "148 SMs x 128 FP32 lanes x 2 x SM clock under load"}
    else:
        ach = d["bytes"] / (d["ms"] * 1e-3) / 1e9
        roof = {"kernel": dom, "bound": "hbm", "achieved": ach, "peak": pk["hbm"], "unit": "GB/s",
                "frac": ach / pk["hbm"], "traffic": profiled_traffic(cfgname, dom), "peak_source": f"{pk['src']} copy bandwidth"}
    tr = roof.get("traffic")
    if isinstance(tr, dict):          # numeric per-launch DRAM bytes of the committed ncu capture + which launch it was
        roof["traffic"] = tr["dram_bytes_per_launch"]
        roof["traffic_from"] = {"launch": tr["launch"], "profile": tr["profile"]}
    roof["avg_launch_ms"] = avg_ms
    roof["launches_per_step"] = d["launches"] / n_aux
    roof["share_of_kernel_time"] = shares.get(dom)
    if dom != "gemm_tc" and aw_tflops:
        roof["aw_contraction"] = {"achieved": aw_tflops, "peak": tc_peak, "frac": aw_tflops / tc_peak, "unit": "TFLOP/s"}

    # ---- NEXT-1: alpha optimisation of the final bound, reported beside the step, not part of it -------
    alpha_opt = None
    if alpha is not None and args.alpha_iters > 0:
        T = args.alpha_iters
        res = {k: torch.empty(B, S, device=dev) for k in ("lb_best", "ub_best", "lb_last", "ub_last")}
        res["verified"] = torch.empty(B, dtype=torch.uint8, device=dev)
        step_device()                                     # (l, u) and the bound at the given alpha
        torch.cuda.synchronize()
        lb_start = io["lb"].clone()
        ms_a = []
        for it in range(3):
            al = {i: a.clone() for i, a in alpha.items()}
            au = {i: a.clone() for i, a in alpha.items()}
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.alpha_ascent_device(io["l"], io["u"], Cd, al, au, xlo, xhi, 0.05, 0.98, T, 1, res)
            e1.record(); e1.synchronize()
            ms_a.append(e0.elapsed_time(e1))
        gain = res["lb_best"] - lb_start
        alpha_opt = {"iters": T, "rule": "sign step, eta 0.05, decay 0.98", "ms_total": min(ms_a), "ms_per_iter": min(ms_a) / (T + 1),
                     "mean_lb_gain": float(gain.mean().item()), "mean_abs_lb_start": float(lb_start.abs().mean().item()),
                     "rows_tightened_frac": float((gain > 0).float().mean().item()),
                     "verified_before": verified, "verified_after": int(res["verified"].sum().item())}
        del res, al, au

    # ---- NEXT-2: beta-CROWN bounds of batched BaB sub-domains, reported beside the step ------------
    bab = None
    if cfgname == "cfg2" and alpha is not None and args.bab_domains > 0 and args.scale == 1:
        bab = measure_bab(wl, ctx, io, args, dev, local)

    # ---- NEXT-3: the same batch with full-CROWN intermediate bounds through the conv layers --------
    conv_crown = None
    if cfgname == "cfg5" and args.scale == 1 and not args.no_conv_crown:
        io2 = ctx.alloc_io(B, S)
        ms_c = []
        for it in range(3):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); ctx.run_device(xlo, xhi, Cd, alpha, 0, io2); e1.record(); e1.synchronize()
            ms_c.append(e0.elapsed_time(e1))
        w_ibp = (io["ub"] - io["lb"]).abs()
        w_cr = (io2["ub"] - io2["lb"]).abs()
        conv_crown = {"ms_per_step": min(ms_c), "properties_per_s": B / (min(ms_c) * 1e-3), "row_chunk": ctx.row_chunk(),
                      "median_final_width_ratio_vs_ibp_intermediates": float((w_cr / w_ibp).median().item()),
                      "verified": int(io2["verified"].sum().item())}
        del io2

    peak_ws = ctx.peak_bytes()
    peak_torch = torch.cuda.max_memory_allocated(dev)
    rc_rows = ctx.row_chunk()
    graph_on = bool(ctx.graph_active())
    cpu = oracle_baseline(wl, cfgname, args.cpu_seconds) if with_cpu else None
    out = {
        "value": world * B / (ms_step * 1e-3), "unit": UNIT, "steps": steps, "ms_per_step": ms_step,
        "config": dict(workload_desc(wl, cfgname), l2="flushed between timed steps (256 MB write)", mem_cap_bytes=cap,
                       row_chunk=rc_rows, stream_weights=bool(args.stream_weights), epi_fusion=not args.no_epi_fusion,
                       graph_replay=graph_on, streamed_layers=len(ctx.streamed_ids),
                       weight_h2d_bytes_per_step=w_h2d_step),
        "verified_last_batch": verified, "aw_tflops": aw_tflops, "aw_flops_per_step": flops_step,
        "peak_hbm_gb": {"workspace_high_water": peak_ws / 1e9, "torch_max_allocated": peak_torch / 1e9,
                        "cudaMemGetInfo_delta": (free0 - free1) / 1e9},
        "kernel_time_shares": shares, "kernel_classes": per_class, "roofline": roof, "cpu_baseline": cpu,
        "e2e": {"value": world * B / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "ms_per_step": ms_e2e, "steps": n_aux},
        "gpu_launches": int(launches_per_step * steps), "gpu_launches_per_step": int(launches_per_step), "clocks": clocks,
        "alpha_opt": alpha_opt, "bab_beta": bab, "conv_crown": conv_crown}
    ctx.close()
    del ctx, xlo, xhi, Cd, alpha, io, flush, wl
    gc.collect()
    torch.cuda.empty_cache()
    torch.cuda.reset_peak_memory_stats(dev)
    return out


def measure_bab(wl, ctx0, io0, args, dev, local):
    """NEXT-2 leg: D sub-domains of the workload's properties (round robin), each the parent's box and intermediate bounds
    (from the step just run, io0) plus `depth` random split decisions on unstable neurons (seeded); one call of
    crown_beta_ascent = T + 1 bound evaluations and T joint projected steps on (alpha, beta) for all sub-domains."""
    import torch
    from paper_2606_09377_b200 import CrownContext
    D, T, depth = args.bab_domains, 10, 8
    S = wl.S
    ctx = CrownContext(wl.net, D, S, device=f"cuda:{local}", mem_cap_bytes=8 << 30)
    g = torch.Generator(device=dev); g.manual_seed(W.SEED_BASE + 777)
    idx = torch.arange(D, device=dev) % wl.B
    lo, hi = wl.box()
    xlo = torch.from_numpy(lo).to(dev)[idx].contiguous(); xhi = torch.from_numpy(hi).to(dev)[idx].contiguous()
    Cd = torch.from_numpy(np.ascontiguousarray(wl.C)).to(dev)[idx].contiguous()
    l = {i: io0["l"][i][idx].contiguous() for i in ctx.relu_ids}
    u = {i: io0["u"][i][idx].contiguous() for i in ctx.relu_ids}
    split = {}
    for i in ctx.relu_ids:        # `depth` splits per sub-domain spread over the layers, on unstable neurons only
        n = ctx.sizes[i]
        pick = torch.rand(D, n, device=dev, generator=g) < (depth / (len(ctx.relu_ids) * n))
        sign = torch.where(torch.rand(D, n, device=dev, generator=g) < 0.5, 1, -1).to(torch.int8)
        split[i] = torch.where(pick & (l[i] < 0) & (u[i] > 0), sign, torch.zeros_like(sign)).contiguous()
    n_split = float(sum(int((s != 0).sum().item()) for s in split.values())) / D
    mk = lambda v: {i: torch.full((D, S, ctx.sizes[i]), v, device=dev) for i in ctx.relu_ids}
    res = {k: torch.empty(D, S, device=dev) for k in ("lb_best", "ub_best", "lb_last", "ub_last")}
    res["verified"] = torch.empty(D, dtype=torch.uint8, device=dev)
    ms = []
    lb0 = None
    for it in range(3):
        al, au, bl, bu = mk(0.5), mk(0.5), mk(0.0), mk(0.0)
        if lb0 is None:       # bounds at the start point (0 iterations)
            ctx.beta_ascent_device(l, u, split, Cd, al, au, bl, bu, xlo, xhi, 0.05, 0.05, 0.98, 0, 1, res)
            torch.cuda.synchronize()
            lb0 = res["lb_best"].clone()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.beta_ascent_device(l, u, split, Cd, al, au, bl, bu, xlo, xhi, 0.05, 0.05, 0.98, T, 1, res)
        e1.record(); e1.synchronize()
        ms.append(e0.elapsed_time(e1))
    gain = res["lb_best"] - lb0
    out = {"domains": D, "iters": T, "splits_per_domain": n_split, "rule": "sign step, eta_alpha = eta_beta = 0.05, decay 0.98",
           "ms_total": min(ms), "ms_per_iter": min(ms) / (T + 1), "domains_per_s": D / (min(ms) * 1e-3),
           "bound_evaluations_per_s": D * (T + 1) / (min(ms) * 1e-3), "mean_lb_gain": float(gain.mean().item()),
           "mean_abs_lb_start": float(lb0.abs().mean().item()), "rows_tightened_frac": float((gain > 0).float().mean().item()),
           "verified_domains": int(res["verified"].sum().item()), "workspace_gb": ctx.peak_bytes() / 1e9}
    ctx.close()
    del ctx, al, au, bl, bu, res, split, l, u
    torch.cuda.empty_cache()
    return out


def run_b200(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the crownb200 hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if args.device_steps_only or args.shard_rows:
        r = measure_config(args.workload, args, args.steps, args.warmup, dev, local, world, None, False)
        if rank == 0:
            print(json.dumps(dict(r, metric=METRIC, n_gpus=world, warmup=args.warmup, higher_is_better=True,
                                  scaling="strong" if args.shard_rows else "weak", data="synthetic",
                                  mode="row-sharded (NEXT-4)" if args.shard_rows else "device-steps-only")))
        if world > 1:
            dist.destroy_process_group()
        return
    tf32_peak = measure_tf32_peak(dev)
    with_cpu = rank == 0 and world == 1 and not args.no_cpu_baseline
    main = measure_config(args.workload, args, args.steps, args.warmup, dev, local, world, tf32_peak, with_cpu)
    per = {}
    if world == 1 and not args.no_per_config and args.scale == 1 and not args.batch:
        for c in ALL_CFGS:
            if c == args.workload:
                continue
            st = {"cfg1": max(args.steps, 20), "cfg2": max(args.steps, 10), "cfg3": min(args.steps, 3),
                  "cfg4": min(args.steps, 5), "cfg5": max(args.steps, 10)}[c]
            r = measure_config(c, args, st, 3, dev, local, world, tf32_peak, with_cpu)
            per[c] = {k: r[k] for k in ("value", "unit", "steps", "ms_per_step", "config", "verified_last_batch", "aw_tflops",
                                        "peak_hbm_gb", "kernel_time_shares", "kernel_classes", "roofline", "cpu_baseline",
                                        "e2e", "gpu_launches_per_step", "clocks", "alpha_opt", "bab_beta", "conv_crown")}
    if rank == 0:
        line = {"metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": main["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32 (3xTF32 products, fp32 accumulate)", "data": "synthetic"}
        for k in ("config", "verified_last_batch", "aw_tflops", "aw_flops_per_step", "peak_hbm_gb", "kernel_time_shares",
                  "kernel_classes", "roofline", "cpu_baseline", "e2e", "gpu_launches", "gpu_launches_per_step", "clocks", "alpha_opt", "bab_beta", "conv_crown"):
            line[k] = main[k]
        line["tf32_dense_peak_tflops"] = tf32_peak
        line["per_config"] = per
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_b200(a)
