#!/usr/bin/env python
"""bench.py -- MoE-layer tokens/s through libef's C ABI, with the grouped-FFN roofline, the H2D link fraction and
the CPU-oracle baseline.  Default workload = BASELINE.json configs[1] (Mixtral-8x7B-shaped prefill, the headline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload mixtral_prefill|mixtral_decode|many_expert_prefill|stack_decode|tiny]

One "step" = one pass of the whole hot path over one batch: per layer visit  [rmsnorm ->] route -> permute ->
cache lookup + real-time correction (on-demand H2D in waves) + grouped SwiGLU FFN -> PLEC prefetch -> combine
[+ residual].  Prefill workloads: 1 visit per step; mixtral_decode: 1 visit of 16 tokens; stack_decode: 32 visits
of 64 tokens.  The cache state carries over from step to step; expert weights stream from the pinned host pool.
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

DUAL_FAMILIES, DUAL_FAMILY_PROB = 2, 0.9     # dual_batch_stack: latent token groups

METRIC = "moe_layer_tokens_per_s"
UNIT = "tokens/s"

# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel (GEMM1) per launch, from the
# committed `ncu --set full` captures (never measured by this script, which never runs under a profiler):
#   mixtral_prefill: profiles/r1f_ffn_prefill_ncu_full.md -- the 6 GEMM1 launches of one steady-state streaming step
#                    (2.0711 GB in all); resident leg: the one launch over all 8 experts (2.0716 GB)
#   mixtral_decode : profiles/r1f_ffn_decode_ncu_full.md  -- 4 GEMM1 launches of a streaming step (three single-expert
#                    waves and one 5-expert wave, 1.8975 GB in all); resident leg: one launch over 7 experts (1.6523 GB)
NCU_TRAFFIC_BYTES = {"mixtral_prefill": 2.0711e9 / 6, "mixtral_decode": 1.8975e9 / 4}
NCU_TRAFFIC_BYTES_RESIDENT = {"mixtral_prefill": 2.0716e9, "mixtral_decode": 1.6523e9}


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
                                          "-lms", "20", "-i", str(self.idx)], stdout=subprocess.PIPE,
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
# workload plumbing shared by both arms (inputs only -- no method arithmetic)
# ---------------------------------------------------------------------------------------------------
def trace_steps_needed(cfg, steps_total: int) -> int:
    return max(1, min(cfg.n_steps, steps_total))


def workload_config(cfg, world, extra=None):
    c = {"workload": cfg.name, "tokens_per_step_per_gpu": cfg.T, "visits_per_step": cfg.n_layers,
         "d_model": cfg.d_model, "d_ff": cfg.d_ff, "n_layers": cfg.n_layers, "n_experts": cfg.n_experts,
         "top_k": cfg.top_k, "cache_slots": cfg.n_slots, "n_shared": cfg.n_shared, "expert_bytes": cfg.expert_bytes,
         "prefetch_horizon": cfg.horizon, "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
         "l2_policy": "inputs larger than L2: every step reads >= 0.69 GB of expert weights from HBM slots that the "
                      "copy stream rewrites, against a 126 MB L2; no explicit flush"}
    if extra:
        c.update(extra)
    return c


# ---------------------------------------------------------------------------------------------------
# the reference arm / cpu_baseline: the oracle as it stands, on host cores, bounded sample
# ---------------------------------------------------------------------------------------------------
def oracle_sample(cfg, n_tokens: int, n_layers: int, cache=None):
    """Time the oracle on a bounded sample of one step: the first n_tokens tokens through the first n_layers
    layers (whole layer each: route, permute, FFN, combine[, rmsnorm + residual]).  Returns tokens/s scaled to a
    whole step (time * L / n_layers), seconds spent, threads used, and a description."""
    import oracle
    L = cfg.n_layers
    n_layers = max(1, min(L, n_layers))
    n_tokens = max(1, min(cfg.T, n_tokens))
    cache = cache if cache is not None else {}
    tr = wl.routing_trace(wl.scaled(cfg, T=cfg.T), 1) if cfg.bias_kind == "trace" else None

    def get(l, e):
        if (l, e) not in cache:
            cache[(l, e)] = wl.expert_weights(cfg, l, e, threads=os.cpu_count() or 8)
        return cache[(l, e)]
    x = wl.activations(cfg, 0)[:n_tokens]
    biases, wrs, needed = [], [], []
    for l in range(n_layers):
        wrs.append(wl.router_weight(cfg, l))
        b = wl.trace_bias(cfg, tr, l)[:n_tokens] if tr is not None else wl.static_router_bias(cfg, l)
        biases.append(b)
        if tr is not None:
            needed.append(sorted(set(int(e) for e in tr.sets[l, :n_tokens].ravel())))
        else:
            needed.append(list(range(cfg.n_experts)))
    # weights are materialised before the clock starts (the GPU arm's sit in pinned memory before its clock too)
    for l in range(n_layers):
        for e in needed[l]:
            get(l, e)
    shared = [[get(l, -1 - s) for s in range(cfg.n_shared)] for l in range(n_layers)]
    t0 = time.perf_counter()
    h = x
    for l in range(n_layers):
        if L > 1:
            u = oracle.round_bf16(oracle.rmsnorm(h, 1e-5))
            ref = oracle.layer_forward(u, wrs[l], biases[l], lambda e, l=l: get(l, e), cfg.top_k, cfg.renorm,
                                       shared=shared[l], res=h)
            h = oracle.round_bf16(ref.out)
        else:
            oracle.layer_forward(h, wrs[l], biases[l], lambda e, l=l: get(l, e), cfg.top_k, cfg.renorm,
                                 shared=shared[l])
    dt = time.perf_counter() - t0
    step_s = dt * L / n_layers
    what = (f"first {n_tokens} of {cfg.T} tokens through the first {n_layers} of {L} layer visit(s) of one step of "
            f"{cfg.name}, whole layer in fp64 ({dt:.1f} s; scaled x{L / n_layers:g} to a step), weights pre-generated, "
            "no host<->device traffic, no cache")
    return n_tokens / step_s, dt, oracle.num_threads(), what


def oracle_sample_dual(cfg, n_tokens: int, n_layers: int, cache=None):
    """dual_batch_stack: the oracle on the first n_tokens tokens of incoming batch 0 of step 0 through the first
    n_layers layers (unscheduled order: the layer result does not depend on the batching)."""
    import oracle
    L = cfg.n_layers
    n_layers = max(1, min(L, n_layers))
    n_tokens = max(1, min(cfg.T, n_tokens))
    cache = cache if cache is not None else {}
    tr = wl.dual_batch_trace(cfg, 1, DUAL_FAMILIES, DUAL_FAMILY_PROB)
    bias = wl.bias_from_sets(cfg, tr.sets[0])[:n_tokens]
    x = wl.normal_bf16(cfg.seed, "x.dual.step0.rank0", (2 * cfg.T, cfg.d_model), 1.0)[:n_tokens]

    def get(l, e):
        if (l, e) not in cache:
            cache[(l, e)] = wl.expert_weights(cfg, l, e, threads=os.cpu_count() or 8)
        return cache[(l, e)]
    wrs = [wl.router_weight(cfg, l) for l in range(n_layers)]
    for l in range(n_layers):
        for e in sorted(set(int(v) for v in tr.sets[0][:n_tokens, l].ravel())):
            get(l, e)
    t0 = time.perf_counter()
    h = x
    for l in range(n_layers):
        u = oracle.round_bf16(oracle.rmsnorm(h, 1e-5))
        ref = oracle.layer_forward(u, wrs[l], bias[:, l], lambda e, l=l: get(l, e), cfg.top_k, cfg.renorm, res=h)
        h = oracle.round_bf16(ref.out)
    dt = time.perf_counter() - t0
    step_s = dt * L / n_layers
    what = (f"first {n_tokens} tokens of incoming batch 0 of step 0 of {cfg.name} through the first {n_layers} of {L} "
            f"layers, whole layer in fp64 ({dt:.1f} s; scaled x{L / n_layers:g}), weights pre-generated, no cache, no scheduler")
    return n_tokens / step_s, dt, oracle.num_threads(), what


def ref_sample_size(cfg, args):
    """Bounded oracle sample: ~10-30 s of CPU work on a 16-core host."""
    n_tok = args.ref_tokens if args.ref_tokens > 0 else {"mixtral_prefill": 256, "many_expert_prefill": 1024, "switch_prefill": 4096}.get(cfg.name, cfg.T)
    n_lay = args.ref_layers if args.ref_layers > 0 else (2 if cfg.n_layers > 1 else 1)
    return n_tok, n_lay


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    cfg = wl.CONFIGS[args.workload]
    n_tok, n_lay = ref_sample_size(cfg, args)
    cache = {}
    vals = []
    sample = oracle_sample_dual if cfg.name == "dual_batch_stack" else oracle_sample
    for i in range(args.warmup + args.steps):
        v, dt, cores, what = sample(cfg, n_tok, n_lay, cache)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals])) * 1e3
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, world),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
class Driver:
    """Owns one MoELayerRunner plus the step inputs of a workload; step(i) = one pass of the whole hot path
    (n_layers visits) over batch i.  Sequencing only: every step of the path runs in libef's kernels."""

    def __init__(self, cfg, dev, x_stream: str, steps_total: int, phys_experts: int = 0, log=lambda *_: None,
                 policy: str = "plec"):
        import torch
        from paper_2410_17954_b200 import MoELayerRunner
        from paper_2410_17954_b200.layer import bf16_tensor_from_bits
        self.torch, self.cfg, self.dev = torch, cfg, dev
        L, E, T, d = cfg.n_layers, cfg.n_experts, cfg.T, cfg.d_model
        self.runner = r = MoELayerRunner(L, E, cfg.top_k, d, cfg.d_ff, cfg.n_slots, cfg.n_shared, T, cfg.horizon,
                                         cfg.renorm, device=dev.index, expert_kind=1 if cfg.expert_kind == "relu" else 0)
        # cache policy arm: the paper's PLEC, the two LRU baselines, or "prefetch every expert of the
        # next layer" = PLEC fed an all-ones predicted path one visit ahead
        r.ctx.ef_set_cache_policy("plec" if policy == "next_layer_all" else policy)
        threads = os.cpu_count() or 8
        n_total = L * E
        self.phys = phys_experts if 0 < phys_experts < n_total else 0
        gen_cfg = wl.scaled(cfg, phys_experts=self.phys)
        t0 = time.perf_counter()
        for l in range(L):
            r.set_router(l, wl.router_weight(cfg, l), wl.static_router_bias(cfg, l))
            for e in range(E):
                g = l * E + e
                if self.phys and g >= self.phys:
                    src = g % self.phys
                    r.ctx.ef_host_expert_alias(l, e, src // E, src % E)
                else:
                    r.register_expert(l, e, *wl.expert_weights(gen_cfg, l, e, threads=threads))
            for s in range(cfg.n_shared):
                r.register_expert(l, -1 - s, *wl.expert_weights(cfg, l, -1 - s, threads=threads))
            if L > 1 and (l % 4 == 3):
                log(f"registered layers 0..{l} ({time.perf_counter() - t0:.0f} s)")
        # step inputs
        self.is_trace = cfg.bias_kind == "trace"
        self.ts = trace_steps_needed(cfg, steps_total) if self.is_trace else 1
        xs = [wl.normal_bf16(cfg.seed, f"x.step{s}.{x_stream}", (T, d), 1.0) for s in range(self.ts)]
        self.x_pin = bf16_tensor_from_bits(np.stack(xs), pin=True)              # [ts, T, d]
        self.x_dev = self.x_pin.to(dev)
        self.x_stage = torch.empty((T, d), dtype=torch.bfloat16, device=dev)    # e2e: per-step H2D target
        self.out = torch.empty((T, d), dtype=torch.bfloat16, device=dev)
        self.hbuf = [torch.empty((T, d), dtype=torch.bfloat16, device=dev) for _ in range(2)]
        self.out_pin = torch.empty((T, d), dtype=torch.bfloat16).pin_memory()
        self.nv = self.ts * L
        if self.is_trace:
            self.trace = wl.routing_trace(cfg, self.ts)
            b = np.stack([wl.trace_bias(cfg, self.trace, v) for v in range(self.nv)])   # [nv, T, E] fp32
            self.bias_pin = torch.from_numpy(b).pin_memory()
            self.bias_dev = self.bias_pin.to(dev)
            self.bias_stage = torch.empty((L, T, E), dtype=torch.float32, device=dev)
            self.look = L if cfg.horizon <= 0 else cfg.horizon
            self.pred = self.trace.predicted
            if policy == "next_layer_all":
                self.pred = np.ones_like(self.pred)
        else:
            self.look = 1
            self.pred = np.ones((1, E), np.uint8)      # replaced by the gate's own active set after warm-up
        self.visit = 0
        r.ctx.ef_cache_prefetch(-1, self.window(-1))

    def window(self, v):
        """Predicted batch-level path rows for visits v+1 .. v+look (the supplied predictor output)."""
        if not self.is_trace:
            return self.pred
        idx = [(v + 1 + j) % self.nv for j in range(self.look)]
        return np.ascontiguousarray(self.pred[idx])

    def adopt_gate_prediction(self):
        """Prefill workloads re-run the same batch every step: the predicted path of the next step is the active
        set the gate produced on this one (read back once, after warm-up)."""
        if not self.is_trace:
            self.torch.cuda.synchronize()
            self.pred = (self.runner.counts.cpu().numpy() > 0).astype(np.uint8)[None, :]

    def step(self, e2e: bool):
        torch, cfg, r = self.torch, self.cfg, self.runner
        L = cfg.n_layers
        s = (self.visit // L) % self.ts
        if e2e:
            self.x_stage.copy_(self.x_pin[s], non_blocking=True)
            x = self.x_stage
            if self.is_trace:
                self.bias_stage.copy_(self.bias_pin[s * L:(s + 1) * L], non_blocking=True)
        else:
            x = self.x_dev[s]
        h = x
        for l in range(L):
            v = self.visit
            tb = None
            if self.is_trace:
                tb = self.bias_stage[l] if e2e else self.bias_dev[v % self.nv]
            dst = self.out if l == L - 1 else self.hbuf[l & 1]
            r.visit(v, h, dst, token_bias=tb, predicted_next=self.window(v), residual=h if L > 1 else None,
                    pre_norm_eps=1e-5 if L > 1 else None)
            h = dst
            self.visit += 1
        if e2e:
            self.out_pin.copy_(self.out, non_blocking=True)
            torch.cuda.current_stream().synchronize()      # the caller reads the result

    def io_bytes(self):
        cfg = self.cfg
        h2d = cfg.T * cfg.d_model * 2 + (cfg.n_layers * cfg.T * cfg.n_experts * 4 if self.is_trace else 0)
        return h2d, cfg.T * cfg.d_model * 2

    def close(self):
        self.runner.close()


def measure_pinned_h2d(dev, nbytes: int, reps: int = 10) -> float:
    """Pinned host -> device copy bandwidth of this box (GB/s): cudaMemcpyAsync of one expert-sized buffer and of a
    1 GiB buffer on an otherwise idle device (the caller drains the library's copy stream first), best of reps,
    CUDA events."""
    import torch
    best = 0.0
    for n in (nbytes, 1 << 30):
        src = torch.empty(n, dtype=torch.uint8).pin_memory()
        src.zero_()
        dst = torch.empty(n, dtype=torch.uint8, device=dev)
        torch.cuda.synchronize()
        for _ in range(reps + 1):
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            e0.record(); dst.copy_(src, non_blocking=True); e1.record(); e1.synchronize()
            best = max(best, n / (e0.elapsed_time(e1) * 1e-3) / 1e9)
        del src, dst
    return best


def run_ours(args):
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    rank, local, world = dist_init("nccl")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    cfg = wl.CONFIGS[args.workload]
    plan = replica_plan(rank, world, cfg.T)
    peaks = measured_peaks()
    log = (lambda m: print(f"[bench] {m}", file=sys.stderr, flush=True)) if rank == 0 else (lambda m: None)

    # host memory check for the pinned pool (cfg 5: 90 GB); alias onto fewer physical buffers if it cannot fit
    phys = args.phys_experts
    need = cfg.n_layers * cfg.n_experts * cfg.expert_bytes
    if phys == 0:
        try:
            avail = int(next(l for l in open("/proc/meminfo") if l.startswith("MemAvailable")).split()[1]) * 1024
        except Exception:
            avail = need * 4
        if need * world > 0.6 * avail:
            phys = max(cfg.n_experts, int(0.5 * avail / world / cfg.expert_bytes))
            log(f"pinned pool of {need / 1e9:.1f} GB does not fit comfortably in {avail / 1e9:.1f} GB of host memory: "
                f"aliasing {cfg.n_layers * cfg.n_experts} logical experts onto {phys} physical buffers")
    steps_total = 2 * (args.steps + args.warmup) + 2
    drv = Driver(cfg, dev, plan["x_stream"], steps_total, phys, log, args.policy)
    runner = drv.runner
    runner.ctx.ef_sync()                 # the warm-up prefetch must not share the link with the peak measurement
    h2d_peak = measure_pinned_h2d(dev, cfg.expert_bytes) if rank == 0 else None

    def timed(e2e, steps, warmup, with_kernel_times=False):
        for _ in range(warmup):
            drv.step(e2e)
        drv.adopt_gate_prediction()
        runner.ctx.ef_sync()
        runner.ctx.ef_cache_reset_stats()               # also clears the copy-busy accumulator
        if with_kernel_times:
            runner.ctx.ef_get_kernel_times(reset=True)
            runner.ctx.ef_set_kernel_timing(True)
        l0 = runner.ctx.ef_launch_count()
        dist_barrier(); torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            drv.step(e2e)
        e1.record()
        runner.ctx.ef_sync()
        torch.cuda.synchronize(); dist_barrier()
        ms = e0.elapsed_time(e1)
        kt = None
        if with_kernel_times:
            kt = runner.ctx.ef_get_kernel_times(reset=True)
            runner.ctx.ef_set_kernel_timing(False)
        st = runner.ctx.ef_cache_get_stats()
        copy_ms = runner.ctx.ef_copy_busy_ms()
        return ms, runner.ctx.ef_launch_count() - l0, kt, st, copy_ms

    sampler = ClockSampler(local)
    sampler.start()
    ms, launches, kt, st, copy_ms = timed(False, args.steps, args.warmup, with_kernel_times=True)
    clocks = sampler.stop()
    ms_max = dist_max(ms, dev)
    value = plan["global_tokens"] * args.steps / (ms_max * 1e-3)

    ms_e2e, _, _, st_e2e, _ = timed(True, args.steps, max(1, args.warmup // 2))
    ms_e2e_max = dist_max(ms_e2e, dev)
    e2e_value = plan["global_tokens"] * args.steps / (ms_e2e_max * 1e-3)
    io_h2d, io_d2h = drv.io_bytes()

    d, f = cfg.d_model, cfg.d_ff
    decode = cfg.T * cfg.top_k / cfg.n_experts < 249 and cfg.name in ("mixtral_decode", "stack_decode")
    fill_peak = None
    if rank == 0 and not decode:
        runner.ctx.ef_sync()
        fill_peak = runner.ctx.ef_debug_tma_fill_gbs(64 << 20, 2000)
    roofline = ffn_roofline(kt, d, f, peaks, decode, "streaming step (one wave of hits + batched waves of misses)",
                            gated=cfg.expert_kind == "swiglu", fill_peak=fill_peak)
    roofline["traffic"] = NCU_TRAFFIC_BYTES.get(cfg.name)
    roofline["traffic_source"] = ("bytes per GEMM1 launch from the committed ncu capture under profiles/ (see NCU_TRAFFIC_BYTES)"
                                  if cfg.name in NCU_TRAFFIC_BYTES else "no ncu capture for this workload")
    roofline["algorithmic_bytes_per_launch"] = ((4.0 if cfg.expert_kind == "swiglu" else 2.0) * d * f * kt["groups"]
                                                + 2.0 * d * kt["rows"] + 2.0 * f * kt["rows"]) / max(1, kt["gemm1_launches"])

    h2d = {"bytes_per_step": st["bytes_h2d"] / args.steps, "loads_per_step": (st["ondemand_loads"] + st["prefetch_issued"]) / args.steps,
           "copy_busy_ms_per_step": copy_ms / args.steps,
           "achieved_gbs": (st["bytes_h2d"] / (copy_ms * 1e-3) / 1e9) if copy_ms > 0 else None,
           "peak_gbs": h2d_peak, "peak_source": "measured in this run on an idle device: pinned->device cudaMemcpyAsync, best of 10 over one "
                          "expert-sized and one 1 GiB buffer",
           "frac": (st["bytes_h2d"] / (copy_ms * 1e-3) / 1e9 / h2d_peak) if copy_ms > 0 and h2d_peak else None,
           "gbs_over_step": st["bytes_h2d"] / (ms * 1e-3) / 1e9,
           "step_ms_lower_bound_from_link": (st["bytes_h2d"] / args.steps / (h2d_peak * 1e9) * 1e3) if h2d_peak else None,
           "copy_overlap": "copies run on the library's copy stream concurrently with the grouped-FFN waves"}
    cache = dict(st)
    cache["hit_ratio"] = st["hits"] / max(1, st["lookups"])

    resident = None
    if rank == 0 and not args.no_resident:
        counts = runner.counts.cpu().numpy()
        drv.close()
        resident = resident_leg(cfg, counts, peaks, dev, args, decode, fill_peak)
    else:
        drv.close()

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_tok, n_lay = ref_sample_size(cfg, args)
        v, dt, cores, what = oracle_sample(cfg, n_tok, n_lay)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": workload_config(cfg, world, {"phys_host_experts": drv.phys or cfg.n_layers * cfg.n_experts,
                                                       "cache_policy": args.policy}),
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": io_h2d + int(st_e2e["bytes_h2d"] / args.steps),
                        "d2h_bytes_per_step": io_d2h, "ms_per_step": ms_e2e_max / args.steps,
                        "expert_loads_per_step": (st_e2e["ondemand_loads"] + st_e2e["prefetch_issued"]) / args.steps,
                        "note": "step inputs (x, per-token router bias) from pinned host memory and out back to pinned "
                                "host memory every step; expert weights stream from the pinned host pool in both legs. "
                                "Trace workloads: this leg continues the routing trace after the device-resident leg, so "
                                "its steps move a different number of experts over the link (expert_loads_per_step here "
                                "against h2d.loads_per_step) and, the step being link-bound, take proportionally long"},
                "gpu_launches": launches, "roofline": roofline, "roofline_resident": resident,
                "h2d": h2d, "cache": cache, "cpu_baseline": cpu_baseline}
        print(json.dumps(line), flush=True)


def run_dual_batch(args):
    """dual_batch_stack: per step TWO incoming batches of T decode tokens go through the Token Scheduler (on the
    predicted routing paths), Reindex, and 2 x L layer visits; the same steps are also run unscheduled (incoming
    batches as they are).  value = tokens/s with the scheduler on."""
    import torch
    from paper_2410_17954_b200 import DualBatchRunner, MoELayerRunner
    from paper_2410_17954_b200.layer import bf16_tensor_from_bits
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    rank, local, world = dist_init("nccl")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    cfg = wl.CONFIGS["dual_batch_stack"]
    L, E, T, d, f = cfg.n_layers, cfg.n_experts, cfg.T, cfg.d_model, cfg.d_ff
    N = 2 * T
    peaks = measured_peaks()
    log = (lambda m: print(f"[bench] {m}", file=sys.stderr, flush=True)) if rank == 0 else (lambda m: None)
    phys = args.phys_experts if args.phys_experts > 0 else 32       # 32 physical host buffers (11 GB) behind 256 logical experts
    runner = MoELayerRunner(L, E, cfg.top_k, d, f, cfg.n_slots, 0, T, cfg.horizon, cfg.renorm, device=dev.index)
    gen_cfg = wl.scaled(cfg, phys_experts=phys)
    threads = os.cpu_count() or 8
    for l in range(L):
        runner.set_router(l, wl.router_weight(cfg, l), None)
        for e in range(E):
            g = l * E + e
            if g >= phys:
                runner.ctx.ef_host_expert_alias(l, e, (g % phys) // E, (g % phys) % E)
            else:
                runner.register_expert(l, e, *wl.expert_weights(gen_cfg, l, e, threads=threads))
    log(f"registered {phys} physical / {L * E} logical experts")
    db = DualBatchRunner(runner, max_iter=8)
    ts = max(1, min(cfg.n_steps, 2 * (args.steps + args.warmup) + 2))
    tr = wl.dual_batch_trace(cfg, ts, DUAL_FAMILIES, DUAL_FAMILY_PROB)
    pred_paths = np.stack([wl.sets_to_paths(tr.pred_sets[s], E) for s in range(ts)])             # [ts, N, L, E] uint8
    bias = np.stack([wl.bias_from_sets(cfg, tr.sets[s]) for s in range(ts)])                     # [ts, N, L, E] fp32
    xs = np.stack([wl.normal_bf16(cfg.seed, f"x.dual.step{s}.rank{rank}", (N, d), 1.0) for s in range(ts)])
    paths_pin = torch.from_numpy(pred_paths).pin_memory(); paths_dev = paths_pin.to(dev)
    bias_pin = torch.from_numpy(bias).pin_memory(); bias_dev = bias_pin.to(dev)
    x_pin = bf16_tensor_from_bits(xs, pin=True); x_dev = x_pin.to(dev)
    paths_stage, bias_stage, x_stage = torch.empty_like(paths_dev[0]), torch.empty_like(bias_dev[0]), torch.empty_like(x_dev[0])
    out = torch.empty((N, d), dtype=torch.bfloat16, device=dev)
    out_pin = torch.empty((N, d), dtype=torch.bfloat16).pin_memory()
    # unscheduled arm: the predicted batch-level rows of the incoming batches [0, T) and [T, 2T) (the baseline's own
    # plumbing, on the host); initial centroids: one seeded draw per step ("random centroid selection")
    rows_off = [np.concatenate([pred_paths[s][b * T:(b + 1) * T].max(axis=0) for b in (0, 1)]) for s in range(ts)]
    cg = wl.stream(cfg.seed, "dual.centroids")
    cents = [tuple(int(v) for v in cg.choice(N, 2, replace=False)) for _ in range(ts)]
    state = {"step": 0}

    def step(sched: bool, e2e: bool):
        s = state["step"] % ts
        if e2e:
            paths_stage.copy_(paths_pin[s], non_blocking=True); bias_stage.copy_(bias_pin[s], non_blocking=True)
            x_stage.copy_(x_pin[s], non_blocking=True)
            p, b, x = paths_stage, bias_stage, x_stage
        else:
            p, b, x = paths_dev[s], bias_dev[s], x_dev[s]
        if sched and not e2e:
            # dual-batch pipeline: this unit's schedule was enqueued on the side stream before the previous
            # unit's decode; pick it up, then enqueue the next unit's before decoding this one
            slot = state["step"] & 1
            if state.get("pending") != state["step"]:
                db.schedule_async(p, cents[s][0], cents[s][1], x, b, slot)
            rows = db.wait_schedule(slot)
            x, b = db.x_re, db.bias_re
            s1 = (state["step"] + 1) % ts
            db.schedule_async(paths_dev[s1], cents[s1][0], cents[s1][1], x_dev[s1], bias_dev[s1], slot ^ 1)
            state["pending"] = state["step"] + 1
        elif sched:
            rows = db.schedule(p, cents[s][0], cents[s][1], x, b)
            x, b = db.x_re, db.bias_re
        else:
            rows = rows_off[s]
        db.run_step(state["step"], rows, x, b, out)
        state["step"] += 1
        if e2e:
            out_pin.copy_(out, non_blocking=True)
            torch.cuda.current_stream().synchronize()

    def timed(sched, e2e, steps, warmup, with_kernel_times=False):
        runner.ctx.ef_sync(); runner.ctx.ef_cache_clear()
        torch.cuda.synchronize()
        state["step"] = 0
        state["pending"] = None
        for _ in range(warmup):
            step(sched, e2e)
        runner.ctx.ef_sync(); runner.ctx.ef_cache_reset_stats()
        if with_kernel_times:
            runner.ctx.ef_get_kernel_times(reset=True); runner.ctx.ef_set_kernel_timing(True)
        l0 = runner.ctx.ef_launch_count()
        dist_barrier(); torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            step(sched, e2e)
        e1.record()
        runner.ctx.ef_sync(); torch.cuda.synchronize(); dist_barrier()
        ms = dist_max(e0.elapsed_time(e1), dev)
        kt = None
        if with_kernel_times:
            kt = runner.ctx.ef_get_kernel_times(reset=True); runner.ctx.ef_set_kernel_timing(False)
        st = runner.ctx.ef_cache_get_stats()
        copy_ms = runner.ctx.ef_copy_busy_ms()
        return {"ms": ms, "launches": runner.ctx.ef_launch_count() - l0, "kt": kt, "st": st, "copy_ms": copy_ms}

    def arm_summary(res, steps):
        st = res["st"]
        return {"tokens_per_s": world * N * steps / (res["ms"] * 1e-3), "ms_per_step": res["ms"] / steps,
                "loads_per_step": (st["ondemand_loads"] + st["prefetch_issued"]) / steps,
                "active_experts_per_visit": st["lookups"] / (steps * 2 * L), "hit_ratio": st["hits"] / max(1, st["lookups"]),
                "bytes_h2d_per_step": st["bytes_h2d"] / steps, "ondemand_loads_per_step": st["ondemand_loads"] / steps}

    runner.ctx.ef_sync()
    h2d_peak = measure_pinned_h2d(dev, cfg.expert_bytes) if rank == 0 else None
    off = timed(False, False, args.steps, args.warmup)
    sampler = ClockSampler(local); sampler.start()
    on = timed(True, False, args.steps, args.warmup, with_kernel_times=True)
    clocks = sampler.stop()
    e2e = timed(True, True, args.steps, max(1, args.warmup // 2))
    # the scheduler call alone (schedule + Reindex + batch-path read-back), CUDA events around 20 calls
    torch.cuda.synchronize()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    objs = []
    e0.record()
    for i in range(20):
        db.schedule(paths_dev[i % ts], cents[i % ts][0], cents[i % ts][1], x_dev[i % ts], bias_dev[i % ts])
        objs.append(db.info.cpu().numpy().copy())
    e1.record(); e1.synchronize()
    sched_us = e0.elapsed_time(e1) / 20 * 1e3
    objs = np.array(objs)
    roofline = ffn_roofline(on["kt"], d, f, peaks, True, "streaming steps with the Token Scheduler on")
    st = on["st"]
    h2d = {"bytes_per_step": st["bytes_h2d"] / args.steps, "copy_busy_ms_per_step": on["copy_ms"] / args.steps,
           "achieved_gbs": st["bytes_h2d"] / (on["copy_ms"] * 1e-3) / 1e9 if on["copy_ms"] > 0 else None, "peak_gbs": h2d_peak,
           "frac": (st["bytes_h2d"] / (on["copy_ms"] * 1e-3) / 1e9 / h2d_peak) if on["copy_ms"] > 0 and h2d_peak else None}
    runner.close()
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_tok, n_lay = ref_sample_size(cfg, args)
        v, dt, cores, what = oracle_sample_dual(cfg, n_tok, n_lay)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what}
    if rank == 0:
        a_on, a_off = arm_summary(on, args.steps), arm_summary(off, args.steps)
        io_h2d = N * d * 2 + N * L * E * 4 + N * L * E
        line = {"metric": METRIC, "value": a_on["tokens_per_s"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": a_on["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": workload_config(cfg, world, {"tokens_per_step_per_gpu": N, "visits_per_step": 2 * L,
                                                       "phys_host_experts": phys, "token_families": DUAL_FAMILIES,
                                                       "family_prob": DUAL_FAMILY_PROB, "scheduler_max_iter": 8}),
                "clocks": clocks,
                "e2e": {"value": world * N * args.steps / (e2e["ms"] * 1e-3), "unit": UNIT,
                        "h2d_bytes_per_step": io_h2d + int(e2e["st"]["bytes_h2d"] / args.steps), "d2h_bytes_per_step": N * d * 2 + 2 * L * E,
                        "ms_per_step": e2e["ms"] / args.steps,
                        "note": "predicted paths, router bias and x from pinned host memory, out back to pinned host memory every step"},
                "gpu_launches": on["launches"], "roofline": roofline, "h2d": h2d,
                "token_scheduler": {"on": a_on, "off": a_off, "speedup": a_on["tokens_per_s"] / a_off["tokens_per_s"],
                                    "schedule_call_us": sched_us,
                                    "pipeline": "dual-batch (P:L189-199): unit n+1 is scheduled on a side stream while unit n "
                                                "decodes (DualBatchRunner.schedule_async / wait_schedule); the e2e leg schedules "
                                                "sequentially because its inputs are staged per step",
                                    "eq5_objective_predicted_paths": {"incoming": float(objs[:, 5].mean()), "scheduled": float(objs[:, 4].mean())},
                                    "kmeans_rounds_mean": float(objs[:, 0].mean()), "converged_frac": float(objs[:, 1].mean())},
                "cache": dict(st, hit_ratio=st["hits"] / max(1, st["lookups"])), "cpu_baseline": cpu_baseline}
        print(json.dumps(line), flush=True)


def ffn_roofline(kt, d, f, peaks, decode, where, gated=True, fill_peak=None):
    """Roofline of the dominant kernel (GEMM1 of the grouped FFN) from the library's per-launch CUDA events.
    gated: SwiGLU experts (GEMM1 contracts against gate AND up: 4 d f FLOP per row); else ReLU experts (2 d f)."""
    t1, t2 = kt["gemm1_ms"] * 1e-3, kt["gemm2_ms"] * 1e-3
    n1, n2 = max(1, kt["gemm1_launches"]), max(1, kt["gemm2_launches"])
    g1 = 4.0 if gated else 2.0
    if decode:
        b1, b2 = g1 * d * f * kt["groups"], 2.0 * d * f * kt["groups"]      # weight bytes read once per active expert
        peak = peaks["hbm_gbs"]
        a1 = b1 / t1 / 1e9 if t1 > 0 else 0.0
        a2 = b2 / t2 / 1e9 if t2 > 0 else 0.0
        return {"bound": "hbm", "kernel": f"ffn_gemm_kernel<swiglu> (GEMM1), {where}", "achieved": a1, "peak": peak,
                "unit": "GB/s", "frac": a1 / peak, "peak_source": f"{peaks['source']} HBM copy bandwidth", "traffic": None,
                "launches": kt["gemm1_launches"], "avg_launch_ms": t1 * 1e3 / n1, "groups_per_launch": kt["groups"] / n1,
                "gemm2": {"achieved": a2, "frac": a2 / peak, "avg_launch_ms": t2 * 1e3 / n2},
                "ffn": {"achieved": (b1 + b2) / (t1 + t2) / 1e9 if t1 + t2 > 0 else 0.0,
                        "frac": (b1 + b2) / (t1 + t2) / 1e9 / peak if t1 + t2 > 0 else 0.0}}
    fl1, fl2 = g1 * d * f * kt["rows"], 2.0 * d * f * kt["rows"]
    peak = peaks["bf16_tflops_sustained"] or peaks["bf16_tflops"]
    a1 = fl1 / t1 / 1e12 if t1 > 0 else 0.0
    a2 = fl2 / t2 / 1e12 if t2 > 0 else 0.0
    # second ceiling: the operand bytes TMA stages into shared memory (from the tile plan) against the measured TMA fill
    # rate of the device -- the L2 -> SM fabric, which is what the prefill GEMM actually runs into
    fab = None
    if fill_peak and kt.get("gemm1_fill_bytes"):
        f1 = kt["gemm1_fill_bytes"] / t1 / 1e9 if t1 > 0 else 0.0
        f2 = kt["gemm2_fill_bytes"] / t2 / 1e9 if t2 > 0 else 0.0
        fab = {"bound": "l2_to_sm", "achieved": f1, "peak": fill_peak, "unit": "GB/s", "frac": f1 / fill_peak,
               "bytes_per_launch": kt["gemm1_fill_bytes"] / n1, "flop_per_fill_byte": fl1 / max(1, kt["gemm1_fill_bytes"]),
               "tflops_at_fill_peak": fl1 / max(1, kt["gemm1_fill_bytes"]) * fill_peak / 1e3,
               "gemm2": {"achieved": f2, "frac": f2 / fill_peak, "flop_per_fill_byte": fl2 / max(1, kt["gemm2_fill_bytes"])},
               "peak_source": "measured in this run: ef_debug_tma_fill_gbs, every SM streaming 32 KB TMA boxes out of a "
                              "64 MB L2-resident region"}
    return {"bound": "tensor", "l2_to_sm": fab, "kernel": f"ffn_gemm_kernel<swiglu> (GEMM1), {where}", "achieved": a1, "peak": peak,
            "unit": "TFLOP/s", "frac": a1 / peak,
            "peak_source": f"{peaks['source']} bf16 sustained (kernel timed inside a long step)", "traffic": None,
            "launches": kt["gemm1_launches"], "avg_launch_ms": t1 * 1e3 / n1, "rows_per_launch": kt["rows"] / n1,
            "gemm2": {"achieved": a2, "frac": a2 / peak, "avg_launch_ms": t2 * 1e3 / n2},
            "ffn": {"achieved": (fl1 + fl2) / (t1 + t2) / 1e12 if t1 + t2 > 0 else 0.0,
                    "frac": (fl1 + fl2) / (t1 + t2) / 1e12 / peak if t1 + t2 > 0 else 0.0}}


def resident_leg(cfg, counts, peaks, dev, args, decode, fill_peak=None):
    """The grouped FFN alone with every active expert of one visit resident (kernel-only roofline): one launch
    pair over all groups, timed by the library's CUDA events on the compute stream, weights > L2."""
    import torch
    from paper_2410_17954_b200 import EfContext
    E = cfg.n_experts
    ctx = EfContext(1, E, cfg.top_k, cfg.d_model, cfg.d_ff, E, 0, cfg.T, 0, dev.index,
                    1 if cfg.expert_kind == "relu" else 0)
    threads = os.cpu_count() or 8
    for e in range(E):
        ctx.ef_host_expert_register(0, e, *wl.expert_weights(cfg, 0, e, threads=threads))
    ctx.ef_cache_prefetch(-1, np.ones((1, E), np.uint8))
    slot_of = {g: s for s, g in enumerate(ctx.ef_cache_snapshot())}
    offs = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    R = int(offs[-1])
    x_perm = torch.randn((R, cfg.d_model), device=dev, dtype=torch.float32).to(torch.bfloat16)
    y = torch.empty((R, cfg.d_model), dtype=torch.bfloat16, device=dev)
    act = [e for e in range(E) if counts[e] > 0]
    rb, rw, sl = [int(offs[e]) for e in act], [int(counts[e]) for e in act], [slot_of[e] for e in act]
    # when the active experts' weights fit in L2 (cfg 4: 64 x 17 MB > 126 MB still; tiny: no) flush between launches
    flush = None
    if len(act) * cfg.expert_bytes < 512e6:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ctx.ef_sync()
    for _ in range(3):
        ctx.ef_expert_ffn_grouped_resident(x_perm, rb, rw, sl, y)
    ctx.ef_sync()
    ctx.ef_set_kernel_timing(True)
    ctx.ef_get_kernel_times(reset=True)
    n = max(5, args.steps)
    for _ in range(n):
        if flush is not None:
            flush.zero_()
        ctx.ef_expert_ffn_grouped_resident(x_perm, rb, rw, sl, y)
    kt = ctx.ef_get_kernel_times(reset=True)
    res = ffn_roofline(kt, cfg.d_model, cfg.d_ff, dict(peaks, bf16_tflops_sustained=None), decode,
                       "all active experts of one visit resident, one launch over all groups",
                       gated=cfg.expert_kind == "swiglu", fill_peak=fill_peak)
    if not decode:
        res["peak_source"] = f"{peaks['source']} bf16 burst (kernel timed alone)"
    res["traffic"] = NCU_TRAFFIC_BYTES_RESIDENT.get(cfg.name)
    res["rows_per_expert"] = [int(c) for c in counts]
    res["l2"] = "256 MB flush write between launches" if flush is not None else "weights exceed L2 between launches"
    ctx.close()
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="mixtral_prefill", choices=sorted(wl.CONFIGS))
    ap.add_argument("--ref-tokens", type=int, default=0, help="tokens in the bounded oracle sample (0 = per-workload default)")
    ap.add_argument("--ref-layers", type=int, default=0, help="layer visits in the bounded oracle sample (0 = default)")
    ap.add_argument("--phys-experts", type=int, default=0,
                    help="alias the logical experts onto this many physical pinned host buffers (0 = one per expert "
                         "if host memory allows)")
    ap.add_argument("--horizon", type=int, default=None,
                    help="override the workload's prefetch horizon H in visits (<= 0: as far as the supplied path reaches; R10)")
    ap.add_argument("--policy", default="plec", choices=["plec", "lru", "layer_lru", "next_layer_all"],
                    help="cache policy arm: the paper's PLEC (default), on-demand LRU over the pool, LRU inside a per-layer "
                         "share, or PLEC prefetching every expert of the next layer (the baselines of P:L230 as policy sketches)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-resident", action="store_true")
    args = ap.parse_args()
    if args.horizon is not None:
        wl.CONFIGS[args.workload] = wl.scaled(wl.CONFIGS[args.workload], horizon=args.horizon)
    if args.policy == "next_layer_all":
        wl.CONFIGS[args.workload] = wl.scaled(wl.CONFIGS[args.workload], horizon=1)
    if args.impl == "reference":
        run_reference(args)
    elif args.workload == "dual_batch_stack":
        run_dual_batch(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
