#!/usr/bin/env python
"""bench.py -- MoE-layer tokens/s on the BASELINE.json headline workload (Mixtral-8x7B-shaped prefill,
configs[1]) through libef's C ABI, with the grouped-GEMM roofline and the CPU-oracle baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

One "step" = one pass of the whole hot path over one batch: route -> permute -> cache lookup + real-time
correction (on-demand H2D in waves) + grouped SwiGLU FFN -> PLEC prefetch -> combine.  With cache capacity
4 of 8 experts and all 8 active, every step streams 4 experts (1.41 GB) from pinned host memory.
N > 1 (torchrun): independent data-parallel replicas, one per GPU, no data-path collective (weak scaling).
"""
from __future__ import annotations

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

import workloads as wl  # noqa: E402

METRIC = "moe_layer_tokens_per_s"
UNIT = "tokens/s"


# ---------------------------------------------------------------------------------------------------
# distributed plumbing (replicas only; works on gloo for the CPU tests)
# ---------------------------------------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def dist_init(backend: str):
    import torch.distributed as dist
    rank, local, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local, world


def dist_barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def dist_max(value: float, device="cpu") -> float:
    """max over ranks of a per-rank device time (never wall clock)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return value
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def dist_sum(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return value
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def replica_plan(rank: int, world: int, tokens_per_replica: int) -> dict:
    """Which batch a rank works on: replicas share weights (same seed) and draw their own activations."""
    return {"rank": rank, "world": world, "tokens": tokens_per_replica, "x_stream": f"rank{rank}",
            "global_tokens": tokens_per_replica * world}


# ---------------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows = []
        self.proc = None
        self.idx = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.idx)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, col in (("hw_slowdown", 5), ("hw_thermal_slowdown", 6), ("sw_thermal_slowdown", 7),
                              ("sw_power_cap", 8)):
                if len(r) > col and r[col].lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------
# peaks
# ---------------------------------------------------------------------------------------------------
def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"bf16_tflops": d["bf16_tflops"], "bf16_tflops_sustained": d.get("bf16_tflops_sustained"),
                "hbm_gbs": d["hbm_gbs"], "source": "measured"}
    return {"bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "hbm_gbs": 6650.0, "source": "fallback"}


# ---------------------------------------------------------------------------------------------------
# the reference arm / cpu_baseline: the oracle as it stands, on host cores, bounded sample
# ---------------------------------------------------------------------------------------------------
def oracle_sample(cfg, n_tokens: int, experts=None):
    """Time the oracle's whole layer on the first n_tokens tokens of the workload."""
    import oracle
    x = wl.activations(cfg)[:n_tokens]
    wr = wl.router_weight(cfg)
    bias = wl.static_router_bias(cfg)
    cache = experts if experts is not None else {}

    def get(e):
        if e not in cache:
            cache[e] = wl.expert_weights(cfg, 0, e)
        return cache[e]
    # weights are materialised before the clock starts (the GPU arm's are resident in pinned memory too)
    for e in range(cfg.n_experts):
        get(e)
    shared = [wl.expert_weights(cfg, 0, -1 - s) for s in range(cfg.n_shared)]
    t0 = time.perf_counter()
    oracle.layer_forward(x, wr, bias, get, cfg.top_k, cfg.renorm, shared=shared)
    dt = time.perf_counter() - t0
    return n_tokens / dt, dt, oracle.num_threads()


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    cfg = wl.CONFIGS[args.workload]
    n = args.ref_tokens
    experts = {}
    vals = []
    for i in range(args.warmup + args.steps):
        v, dt, cores = oracle_sample(cfg, n, experts)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals])) * 1e3
    sample = f"first {n} of {cfg.T} tokens of {cfg.name} per step, whole layer in fp64, weights pre-generated"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, world),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(cfg, world):
    return {"workload": cfg.name, "tokens_per_step_per_gpu": cfg.T, "d_model": cfg.d_model, "d_ff": cfg.d_ff,
            "n_experts": cfg.n_experts, "top_k": cfg.top_k, "cache_slots": cfg.n_slots, "n_shared": cfg.n_shared,
            "expert_bytes": cfg.expert_bytes, "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
            "l2_policy": "per-step weight traffic (>= 1.4 GB) exceeds the 126 MB L2; no explicit flush"}


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2410_17954_b200 import MoELayerRunner
    from paper_2410_17954_b200.layer import bf16_tensor_from_bits

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    rank, local, world = dist_init("nccl")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    cfg = wl.CONFIGS[args.workload]
    plan = replica_plan(rank, world, cfg.T)
    peaks = measured_peaks()

    runner = MoELayerRunner(cfg.n_layers, cfg.n_experts, cfg.top_k, cfg.d_model, cfg.d_ff, cfg.n_slots, cfg.n_shared,
                            cfg.T, cfg.horizon, cfg.renorm, device=local)
    runner.set_router(0, wl.router_weight(cfg), wl.static_router_bias(cfg))
    for e in range(cfg.n_experts):
        runner.register_expert(0, e, *wl.expert_weights(cfg, 0, e, threads=os.cpu_count() or 8))
    for s in range(cfg.n_shared):
        runner.register_expert(0, -1 - s, *wl.expert_weights(cfg, 0, -1 - s))
    x_bits = wl.normal_bf16(cfg.seed, f"x.step0.{plan['x_stream']}", (cfg.T, cfg.d_model), 1.0)
    x_pin = bf16_tensor_from_bits(x_bits, pin=True)
    x_dev = x_pin.to(dev)
    out = torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16, device=dev)
    out_pin = torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16).pin_memory()
    # the supplied predicted path: every expert active (true for this workload: T*k >> E); cold cache + warm-up
    predicted = np.ones((1, cfg.n_experts), np.uint8)
    runner.ctx.ef_cache_prefetch(-1, predicted)

    visit = [0]

    def step_device():
        runner.visit(visit[0], x_dev, out, predicted_next=predicted)
        visit[0] += 1

    def step_e2e():
        x_dev.copy_(x_pin, non_blocking=True)
        runner.visit(visit[0], x_dev, out, predicted_next=predicted)
        out_pin.copy_(out, non_blocking=True)
        torch.cuda.current_stream().synchronize()      # the caller reads the result
        visit[0] += 1

    def timed(fn, steps, warmup, with_kernel_times=False):
        for _ in range(warmup):
            fn()
        runner.ctx.ef_sync()
        if with_kernel_times:
            runner.ctx.ef_get_kernel_times(reset=True)
            runner.ctx.ef_set_kernel_timing(True)
        l0 = runner.ctx.ef_launch_count()
        st0 = runner.ctx.ef_cache_get_stats()
        dist_barrier(); torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        runner.ctx.ef_sync()
        torch.cuda.synchronize(); dist_barrier()
        ms = e0.elapsed_time(e1)
        kt = None
        if with_kernel_times:
            kt = runner.ctx.ef_get_kernel_times(reset=True)
            runner.ctx.ef_set_kernel_timing(False)
        st1 = runner.ctx.ef_cache_get_stats()
        return ms, runner.ctx.ef_launch_count() - l0, kt, {k: st1[k] - st0[k] for k in st1}

    sampler = ClockSampler(local)
    sampler.start()
    ms, launches, kt, dstats = timed(step_device, args.steps, args.warmup, with_kernel_times=True)
    clocks = sampler.stop()
    ms_max = dist_max(ms, dev)
    value = plan["global_tokens"] * args.steps / (ms_max * 1e-3)

    ms_e2e, _, _, _ = timed(step_e2e, args.steps, max(1, args.warmup // 2))
    ms_e2e_max = dist_max(ms_e2e, dev)
    e2e_value = plan["global_tokens"] * args.steps / (ms_e2e_max * 1e-3)
    io_bytes = cfg.T * cfg.d_model * 2

    # roofline of the dominant kernel (GEMM1: gate/up projection + SwiGLU), launches of the timed region
    d, f = cfg.d_model, cfg.d_ff
    flops1 = 4.0 * d * f * kt["rows"]
    flops2 = 2.0 * d * f * kt["rows"]
    ach1 = flops1 / (kt["gemm1_ms"] * 1e-3) / 1e12 if kt["gemm1_ms"] > 0 else 0.0
    ach2 = flops2 / (kt["gemm2_ms"] * 1e-3) / 1e12 if kt["gemm2_ms"] > 0 else 0.0
    peak = peaks["bf16_tflops_sustained"] or peaks["bf16_tflops"]
    roofline = {"bound": "tensor", "kernel": "ffn_gemm_kernel<swiglu> (GEMM1, streaming step: 1 wave of hits + 1 wave per miss)",
                "achieved": ach1, "peak": peak, "unit": "TFLOP/s", "frac": ach1 / peak,
                "peak_source": f"{peaks['source']} bf16 sustained (kernel timed inside a long step)",
                "traffic": None, "launches": kt["gemm1_launches"], "avg_launch_ms": kt["gemm1_ms"] / max(1, kt["gemm1_launches"]),
                "gemm2": {"achieved": ach2, "frac": ach2 / peak, "avg_launch_ms": kt["gemm2_ms"] / max(1, kt["gemm2_launches"])}}

    # kernel-only leg: all experts resident (second context with E slots), the grouped GEMM alone
    resident = None
    if rank == 0 and not args.no_resident:
        resident = resident_leg(cfg, runner, peaks, dev, args)

    h2d = {"bytes_per_step": dstats["bytes_h2d"] / args.steps,
           "gbs_over_step": dstats["bytes_h2d"] / (ms * 1e-3) / 1e9}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n = args.ref_tokens
        v, dt, cores = oracle_sample(cfg, n)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"first {n} of {cfg.T} tokens, whole layer in fp64, {dt:.1f} s, weights pre-generated, "
                                  "no host<->device traffic"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": workload_config(cfg, world), "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": io_bytes + int(h2d["bytes_per_step"]),
                        "d2h_bytes_per_step": io_bytes, "ms_per_step": ms_e2e_max / args.steps,
                        "note": "x from pinned host and out back to pinned host every step; expert weights stream "
                                "from the pinned host pool in both legs"},
                "gpu_launches": launches, "roofline": roofline, "roofline_resident": resident,
                "h2d": h2d, "cache": dstats, "cpu_baseline": cpu_baseline}
        print(json.dumps(line), flush=True)
    runner.close()


def resident_leg(cfg, runner, peaks, dev, args):
    """Grouped FFN alone with every needed expert resident: the prefill tensor-core roofline."""
    import torch
    from paper_2410_17954_b200 import EfContext
    counts = runner.counts.cpu().numpy()
    runner.close()                                   # free the streaming arena before allocating E slots
    E = cfg.n_experts
    ctx = EfContext(1, E, cfg.top_k, cfg.d_model, cfg.d_ff, E, 0, cfg.T, 0, dev.index)
    for e in range(E):
        ctx.ef_host_expert_register(0, e, *wl.expert_weights(cfg, 0, e, threads=os.cpu_count() or 8))
    ctx.ef_cache_prefetch(-1, np.ones((1, E), np.uint8))
    slot_of = {g: s for s, g in enumerate(ctx.ef_cache_snapshot())}
    offs = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    R = int(offs[-1])
    x_perm = torch.randn((R, cfg.d_model), device=dev, dtype=torch.float32).to(torch.bfloat16)
    y = torch.empty((R, cfg.d_model), dtype=torch.bfloat16, device=dev)
    act = [e for e in range(E) if counts[e] > 0]
    rb, rw, sl = [int(offs[e]) for e in act], [int(counts[e]) for e in act], [slot_of[e] for e in act]
    ctx.ef_sync()
    for _ in range(3):
        ctx.ef_expert_ffn_grouped_resident(x_perm, rb, rw, sl, y)
    ctx.ef_sync()
    ctx.ef_set_kernel_timing(True)
    ctx.ef_get_kernel_times(reset=True)
    n = max(5, args.steps)
    for _ in range(n):
        ctx.ef_expert_ffn_grouped_resident(x_perm, rb, rw, sl, y)
    kt = ctx.ef_get_kernel_times(reset=True)
    d, f = cfg.d_model, cfg.d_ff
    t1, t2 = kt["gemm1_ms"] / n, kt["gemm2_ms"] / n
    fl1, fl2 = 4.0 * d * f * R, 2.0 * d * f * R
    peak = peaks["bf16_tflops"]
    res = {"rows": R, "rows_per_expert": [int(c) for c in counts], "gemm1_ms": t1, "gemm2_ms": t2,
           "gemm1_tflops": fl1 / t1 / 1e9, "gemm2_tflops": fl2 / t2 / 1e9,
           "ffn_tflops": (fl1 + fl2) / (t1 + t2) / 1e9, "peak": peak, "unit": "TFLOP/s",
           "frac": (fl1 + fl2) / (t1 + t2) / 1e9 / peak, "peak_source": f"{peaks['source']} bf16 burst",
           "note": "true ragged rows, padding not counted; weights (2.8 GB) exceed L2 between launches"}
    ctx.close()
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="mixtral_prefill", choices=sorted(wl.CONFIGS))
    ap.add_argument("--ref-tokens", type=int, default=256, help="tokens in the bounded oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-resident", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
