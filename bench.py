#!/usr/bin/env python
"""bench.py -- one JSON line for the CROWN hot path on B200 (contract: DESIGN.md sec. "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl b200|reference]

A "step" is one pass of the whole hot path (IBP -> CROWN intermediate bounds for every ReLU -> alpha-CROWN
final bound -> concretisation -> verdict) over one batch of synthetic input.
Default workload = BASELINE.json configs[1]: MNIST-FC-shaped MLP 784-(256x6)-10, 64 properties x 3 eps
(192 properties per step), 9 margin specs each, alpha ~ U[0,1].  Inputs are seeded and synthetic
(workloads.py); they stand in for the paper's VNN-COMP MNIST-FC instances, which are not reproduced.

value  : properties/s, device-timed (CUDA events on the launching stream), inputs resident in HBM.
e2e    : same metric through crown_run_host: pinned HOST buffers, H2D of x_lo/x_hi/C/alpha and D2H of
         lb/ub/verified inside the timed region.
Multi-GPU (torchrun): properties are independent, every rank runs its own batch (weak scaling), no
data-path collective; time = max over ranks.
--impl reference: the float64 CPU oracle (oracle/) as it stands, on a bounded sample per step.
"""
from __future__ import annotations

import argparse
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
TF32_OVER_BF16 = 1.1 / 2.25          # nominal dense ratio (B200_PROFILING.md table)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--scale", type=int, default=1, help="width divisor (debug only; 1 = the named config)")
    ap.add_argument("--batch", type=int, default=0, help="override B (debug only)")
    ap.add_argument("--mem-cap-gb", type=float, default=0.0)
    ap.add_argument("--stream-weights", action="store_true",
                    help="layers with >= 2^28 weights are streamed from pinned host memory (a7), not resident")
    ap.add_argument("--no-epi-fusion", action="store_true", help="run the relaxation as its own kernel (debug)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
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


def workload_desc(wl, cfgname):
    return {"workload": f"{cfgname}:{wl.name}", "B": int(wl.B), "S": int(wl.S),
            "eps_set": sorted({round(float(e), 6) for e in wl.eps}), "properties_per_step": int(wl.B),
            "intermediate": wl.intermediate, "alpha": wl.alpha is not None}


def boxes(wl):
    """The (x_lo, x_hi) batches of a step.  Workloads with several eps (cfg2: 64 points x 3 eps) are stacked by
    workloads.stack_eps into ONE batch of per-property radii before this is called (reading G13)."""
    return [wl.box()]


# ------------------------------------------------------------------------------------------------
# oracle legs (cpu_baseline and --impl reference): the ONLY places bench.py executes oracle/
# ------------------------------------------------------------------------------------------------
def oracle_sample(wl, bxs, budget_s, max_props=None):
    """Runs the float64 oracle, as it stands, on properties 0,1,... of the eps batches (round robin) until
    budget_s is spent (at least one property).  Returns (properties done, seconds, threads)."""
    from oracle import crown_oracle as O
    try:
        from threadpoolctl import threadpool_info
        thr = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        thr = os.cpu_count() or 1
    done, t0 = 0, time.perf_counter()
    k = max(1, len({float(e) for e in wl.eps}))          # stacked eps groups: visit them round robin
    per = max(1, wl.B // k)
    order = [(p, 0) for p in sorted(range(wl.B), key=lambda q: (q % per, q // per))]
    for p, e in order:
        lo, hi = bxs[e]
        al = None if wl.alpha is None else [a[p] for a in wl.alpha]
        O.run_property(wl.net, lo[p], hi[p], wl.C[p], al, wl.intermediate)
        done += 1
        if time.perf_counter() - t0 >= budget_s or (max_props and done >= max_props):
            break
    return done, time.perf_counter() - t0, thr


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = int(args.workload[3:])
    wl = W.stack_eps(W.make(cfg, scale=args.scale, B=args.batch or None))
    bxs = boxes(wl)
    # each step = a bounded sample (first `per_step` properties) so K+W steps end within minutes
    n1, t1, thr = oracle_sample(wl, bxs, 0.0, max_props=1)
    per_step = max(1, min(wl.B * len(bxs), int(5.0 / max(t1 / n1, 1e-6))))
    for _ in range(min(args.warmup, 1)):
        oracle_sample(wl, bxs, 1e9, max_props=per_step)
    tot_n, tot_t = 0, 0.0
    for _ in range(args.steps):
        n, t, thr = oracle_sample(wl, bxs, 1e9, max_props=per_step)
        tot_n += n
        tot_t += t
    v = tot_n / tot_t
    sample = f"{per_step} of {wl.B * len(bxs)} properties per step (first ones, eps round robin), float64 numpy"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_desc(wl, args.workload),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": sample},
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


# ------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------
def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_2606_09377_b200 import CrownContext, multi

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the crownb200 hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg = int(args.workload[3:])
    wl = W.stack_eps(W.make(cfg, scale=args.scale, B=args.batch or None))
    bxs = boxes(wl)
    B, S, nE = wl.B, wl.S, len(bxs)
    props_per_step = B * nE
    cap = int(args.mem_cap_gb * (1 << 30))
    if cap == 0 and cfg in (3, 4):
        cap = 64 << 30
    ctx = CrownContext(wl.net, B, S, device=f"cuda:{local}", mem_cap_bytes=cap,
                       stream_weights=int(args.stream_weights), disable_epi_fusion=int(args.no_epi_fusion))
    inter = 1 if wl.intermediate == "ibp" else 0

    # ---- inputs resident in HBM -------------------------------------------------------------------
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    xlo = [t(lo) for lo, _ in bxs]
    xhi = [t(hi) for _, hi in bxs]
    Cd = t(wl.C)
    alpha = None if wl.alpha is None else {i: t(a) for i, a in zip(ctx.relu_ids, wl.alpha)}
    io = ctx.alloc_io(B, S)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def step_device():
        for e in range(nE):
            ctx.run_device(xlo[e], xhi[e], Cd, alpha, inter, io)

    # ---- pinned host buffers for the end-to-end leg ---------------------------------------------------
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_xlo = [pin(lo) for lo, _ in bxs]
    h_xhi = [pin(hi) for _, hi in bxs]
    h_C = pin(wl.C)
    h_alpha = None if wl.alpha is None else [pin(a) for a in wl.alpha]
    h_lb = torch.empty(B, S).pin_memory()
    h_ub = torch.empty(B, S).pin_memory()
    h_ver = torch.empty(B, dtype=torch.uint8).pin_memory()
    h2d = nE * (2 * B * ctx.n0 * 4 + h_C.numel() * 4 + (sum(a.numel() for a in h_alpha) * 4 if h_alpha else 0))
    d2h = nE * (2 * B * S * 4 + B)

    def step_host():
        for e in range(nE):
            ctx.run_host(h_xlo[e].numpy(), h_xhi[e].numpy(), h_C.numpy(),
                         None if h_alpha is None else [a.numpy() for a in h_alpha], wl.intermediate,
                         h_lb.numpy(), h_ub.numpy(), h_ver.numpy())

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, warmup, host_clock=False):
        for _ in range(warmup):
            fn()
        barrier()
        ms = []
        for _ in range(steps):
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
        return multi.max_over_ranks(sum(ms)) / steps       # the job is as slow as its slowest replica

    clk = ClockSampler(local)
    l0 = ctx.launch_count()
    step_device()
    launches_per_step = ctx.launch_count() - l0
    f0 = ctx.gemm_flops()
    clk.start()
    ms_step = timed(step_device, args.steps, max(args.warmup - 1, 0))
    clocks = clk.stop()
    flops_step = (ctx.gemm_flops() - f0) / (args.steps + max(args.warmup - 1, 0))
    w_h2d_step = ctx.h2d_bytes() / (args.steps + max(args.warmup - 1, 0) + 1)
    verified = int(io["verified"].sum().item())      # of the last eps batch
    # end-to-end: host buffers in, host results out, wall clock around the blocking C-ABI call
    ms_e2e = timed(step_host, args.steps, max(args.warmup, 1), host_clock=True)

    # ---- per-kernel-class device times over the same steps (CUDA events around every launch) ------------
    ctx.timing(True)
    for _ in range(args.steps):
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
    # per kernel class: launches per step, mean device time, achieved algorithmic GB/s and TFLOP/s (bytes / flops are the
    # library's own per-launch algorithmic counts)
    per_class = {k: {"launches_per_step": c["launches"] / args.steps, "ms_per_step": c["ms"] / args.steps,
                     "gbs": (c["bytes"] / (c["ms"] * 1e-3) / 1e9) if c["ms"] > 0 and c["bytes"] > 0 else None,
                     "tflops": (c["flops"] / (c["ms"] * 1e-3) / 1e12) if c["ms"] > 0 and c["flops"] > 0 else None}
                 for k, c in classes.items() if c["launches"]}
    d = classes[dom]
    avg_ms = d["ms"] / max(d["launches"], 1)
    if dom == "gemm_tc":
        bf16 = pk["bf16_sustained"] if long_step else pk["bf16"]
        peak = bf16 * TF32_OVER_BF16 / 3.0           # fp32-equivalent: 3 TF32 MMAs per useful product
        ach = d["flops"] / d["launches"] / (avg_ms * 1e-3) / 1e12
        # DRAM bytes per launch from the committed ncu --set full capture of this command (profiles/r1_gemm_tf32x3_cfg2.md:
        # 202 MB read + 70 MB written per N = 256 launch at B = 192; algorithmic 4(2MK + 2KN + MN) = 302 MB, the
        # difference is L2 hits on limbs the relax kernel just wrote); null for workloads without a committed capture
        traffic = 2.72e8 if (cfg == 2 and args.scale == 1 and not args.batch and not args.no_epi_fusion) else None
        roof = {"kernel": "gemm_tf32x3_kernel", "bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                "frac": ach / peak, "traffic": traffic,
                "peak_source": f"{pk['src']} bf16 {'sustained' if long_step else 'burst'} x nominal tf32/bf16 ratio / 3"}
    else:
        ach = d["bytes"] / max(d["launches"], 1) / (avg_ms * 1e-3) / 1e9
        roof = {"kernel": dom, "bound": "hbm", "achieved": ach, "peak": pk["hbm"], "unit": "GB/s",
                "frac": ach / pk["hbm"], "traffic": None, "peak_source": f"{pk['src']} copy bandwidth"}
    roof["avg_launch_ms"] = avg_ms
    roof["launches_per_step"] = d["launches"] / args.steps
    roof["share_of_kernel_time"] = shares.get(dom)
    g = classes["gemm_tc"]
    aw_tflops = (g["flops"] / (g["ms"] * 1e-3) / 1e12) if g["ms"] > 0 else None

    peak_ws = ctx.peak_bytes()
    peak_torch = torch.cuda.max_memory_allocated(dev)

    # ---- CPU baseline: the oracle as it stands, bounded sample, rank 0 only --------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n, secs, thr = oracle_sample(wl, bxs, args.cpu_seconds)
        cpu = {"value": n / secs, "unit": UNIT, "cores": thr, "kind": "oracle",
               "sample": f"first {n} of {props_per_step} properties (eps round robin), {secs:.1f} s, float64 numpy"}

    if rank == 0:
        value = world * props_per_step / (ms_step * 1e-3)
        e2e = world * props_per_step / (ms_e2e * 1e-3)
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32 (3xTF32 products, fp32 accumulate)", "data": "synthetic",
            "config": dict(workload_desc(wl, args.workload), l2="flushed between timed steps (256 MB write)",
                           mem_cap_bytes=cap, stream_weights=bool(args.stream_weights), epi_fusion=not args.no_epi_fusion,
                           streamed_layers=len(ctx.streamed_ids), weight_h2d_bytes_per_step=w_h2d_step),
            "verified_last_batch": verified, "aw_tflops": aw_tflops, "aw_flops_per_step": flops_step,
            "peak_hbm_gb": {"workspace_high_water": peak_ws / 1e9, "torch_max_allocated": peak_torch / 1e9},
            "kernel_time_shares": shares, "kernel_classes": per_class,
            "roofline": roof, "cpu_baseline": cpu,
            "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": ms_e2e},
            "gpu_launches": int(launches_per_step * args.steps), "clocks": clocks}))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_b200(a)
