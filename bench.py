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

# roofline.traffic = dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel per launch, from the committed
# `ncu --set full` captures (this script never runs under a profiler).  profiles/ncu_traffic.json records the numbers
# together with the git blob hash of csrc/ffn_tc.cu they were taken at; when the kernel source has changed since, the
# line says traffic: null, traffic_stale: true instead of quoting a number that no longer describes the code.
def git_blob_hash(path: str) -> str:
    import hashlib
    data = open(path, "rb").read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def ncu_traffic(workload: str, leg: str):
    """(bytes per launch or None, stale flag, source text) for leg in {"in_step", "resident"}."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(path):
        return None, False, "no profiles/ncu_traffic.json"
    rec = json.load(open(path))
    ent = rec.get("workloads", {}).get(workload, {}).get(leg)
    if ent is None:
        return None, False, "no ncu capture of this workload / leg in profiles/ncu_traffic.json"
    cur = git_blob_hash(os.path.join(ROOT, "paper_2410_17954_b200", "csrc", "ffn_tc.cu"))
    if cur != rec.get("ffn_tc_blob"):
        return None, True, f"capture taken at ffn_tc.cu blob {rec.get('ffn_tc_blob', '?')[:12]}, source is now {cur[:12]}"
    return ent["bytes_per_launch"], False, ent.get("source", "profiles/ncu_traffic.json")


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
         "prefetch_horizon": cfg.horizon, "parallelism": f"replicas x{world}" if world > 1 else "single GPU"}
    # expert weights a step reads from HBM slots (every active expert once; the copy stream rewrites the slots it evicts)
    act = min(cfg.n_experts, cfg.T * cfg.top_k) * cfg.n_layers
    c["l2_policy"] = (f"inputs larger than L2: a step reads up to {act} experts x {cfg.expert_bytes / 1e6:.1f} MB = "
                      f"{act * cfg.expert_bytes / 1e9:.2f} GB of weights out of HBM slots against a 126 MB L2; no explicit "
                      "flush in the streaming step (the resident leg flushes when its weights would fit)")
    if extra:
        c.update(extra)
    return c


# ---------------------------------------------------------------------------------------------------
# the reference arm / cpu_baseline: the oracle as it stands, on host cores, bounded sample
# ---------------------------------------------------------------------------------------------------
def oracle_sample(cfg, n_tokens: int, n_layers: int, cache=None, real: str = "double"):
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
            u = oracle.round_bf16(oracle.rmsnorm(h, 1e-5, real=real), real=real)
            ref = oracle.layer_forward(u, wrs[l], biases[l], lambda e, l=l: get(l, e), cfg.top_k, cfg.renorm,
                                       shared=shared[l], res=h, real=real)
            h = oracle.round_bf16(ref.out, real=real)
        else:
            oracle.layer_forward(h, wrs[l], biases[l], lambda e, l=l: get(l, e), cfg.top_k, cfg.renorm,
                                 shared=shared[l], real=real)
    dt = time.perf_counter() - t0
    step_s = dt * L / n_layers
    what = (f"first {n_tokens} of {cfg.T} tokens through the first {n_layers} of {L} layer visit(s) of one step of "
            f"{cfg.name}, whole layer in {'fp64' if real == 'double' else 'fp32'} ({dt:.1f} s; scaled x{L / n_layers:g} to a "
            "step), weights pre-generated, no host<->device traffic, no cache")
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
    real = "float" if args.ref_precision == "fp32" and cfg.name != "dual_batch_stack" else "double"
    sample = oracle_sample_dual if cfg.name == "dual_batch_stack" else (lambda c, t, l, ca: oracle_sample(c, t, l, ca, real=real))
    for i in range(args.warmup + args.steps):
        v, dt, cores, what = sample(cfg, n_tok, n_lay, cache)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals])) * 1e3
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if real == "double" else "f32", "data": "synthetic",
            "config": workload_config(cfg, world, {"phys_host_experts": cfg.n_layers * cfg.n_experts, "cache_policy": args.policy}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what,
                             "precision": "fp64" if real == "double" else "fp32"},
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


def cpu_baseline_block(cfg, args):
    """The oracle as it stands on the host cores, bounded sample: fp64 (the oracle's default, what the parity tests use)
    and the same C file built with -DORC_REAL=float (the fp32 oracle BASELINE.json's north_star describes)."""
    n_tok, n_lay = ref_sample_size(cfg, args)
    cache = {}
    v, dt, cores, what = oracle_sample(cfg, n_tok, n_lay, cache)
    v32, dt32, _, what32 = oracle_sample(cfg, n_tok, n_lay, cache, real="float")
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what, "precision": "fp64",
            "fp32": {"value": v32, "unit": UNIT, "cores": cores, "kind": "oracle", "precision": "fp32", "sample": what32}}


def measure_fill_peak(dev):
    """L2 -> SM fill ceiling of this device, from the DIAGNOSTIC library's probe kernel (ef_diag.h): the
    product library carries no probe.  None when libef_diag.so has not been built."""
    from paper_2410_17954_b200 import EfContext, EfError
    try:
        ctx = EfContext(1, 8, 1, 256, 512, 1, 0, 16, 0, dev.index, 0, diag=True)
    except (EfError, OSError):
        return None
    try:
        return ctx.ef_diag_tma_fill_gbs(64 << 20, 2000)
    finally:
        ctx.close()


def measure_workload(cfg, args, dev, plan, world, peaks, log, steps, warmup, want_e2e=True, want_resident=True, fill_peak=None,
                     sample_clocks=True, local=0, rank=0):
    """One workload through the whole path: device-resident leg (+ per-launch FFN roofline), optional end-to-end leg,
    optional resident-FFN leg.  Returns a dict of the pieces of the JSON line."""
    import torch
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
    steps_total = 2 * (steps + warmup) + 2
    drv = Driver(cfg, dev, plan["x_stream"], steps_total, phys, log, args.policy)
    if args.no_early_release:
        from paper_2410_17954_b200 import EF_OPT_EARLY_RELEASE
        drv.runner.ctx.ef_set_option(EF_OPT_EARLY_RELEASE, 0)
    runner = drv.runner
    runner.ctx.ef_sync()                 # the warm-up prefetch must not share the link with the peak measurement
    h2d_peak = measure_pinned_h2d(dev, cfg.expert_bytes) if rank == 0 else None

    def timed(e2e, n_steps, n_warm, with_kernel_times=False):
        for _ in range(n_warm):
            drv.step(e2e)
        drv.adopt_gate_prediction()
        runner.ctx.ef_sync()
        runner.ctx.ef_cache_reset_stats()               # also clears the copy-busy accumulator
        if with_kernel_times:
            runner.ctx.ef_get_kernel_times(reset=True)
            runner.ctx.ef_get_launch_log(reset=True)
            runner.ctx.ef_set_kernel_timing(True)
        l0 = runner.ctx.ef_launch_count()
        dist_barrier(); torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n_steps):
            drv.step(e2e)
        e1.record()
        runner.ctx.ef_sync()
        torch.cuda.synchronize(); dist_barrier()
        ms = e0.elapsed_time(e1)
        kt = lg = None
        if with_kernel_times:
            kt = runner.ctx.ef_get_kernel_times(reset=True)
            lg = runner.ctx.ef_get_launch_log(reset=True)
            runner.ctx.ef_set_kernel_timing(False)
        st = runner.ctx.ef_cache_get_stats()
        copy_ms = runner.ctx.ef_copy_busy_ms()
        return ms, runner.ctx.ef_launch_count() - l0, kt, lg, st, copy_ms

    sampler = ClockSampler(local) if sample_clocks else None
    if sampler:
        sampler.start()
    ms, launches, kt, lg, st, copy_ms = timed(False, steps, warmup, with_kernel_times=True)
    clocks = sampler.stop() if sampler else None
    ms_max = dist_max(ms, dev)
    value = plan["global_tokens"] * steps / (ms_max * 1e-3)
    res = {"value": value, "ms_per_step": ms_max / steps, "clocks": clocks, "gpu_launches": launches}

    if want_e2e:
        ms_e2e, _, _, _, st_e2e, _ = timed(True, steps, max(1, warmup // 2))
        ms_e2e_max = dist_max(ms_e2e, dev)
        io_h2d, io_d2h = drv.io_bytes()
        res["e2e"] = {"value": plan["global_tokens"] * steps / (ms_e2e_max * 1e-3), "unit": UNIT,
                      "h2d_bytes_per_step": io_h2d + int(st_e2e["bytes_h2d"] / steps), "d2h_bytes_per_step": io_d2h,
                      "ms_per_step": ms_e2e_max / steps,
                      "expert_loads_per_step": (st_e2e["ondemand_loads"] + st_e2e["prefetch_issued"]) / steps,
                      "note": "step inputs (x, per-token router bias) from pinned host memory and out back to pinned "
                              "host memory every step; expert weights stream from the pinned host pool in both legs. "
                              "Trace workloads: this leg continues the routing trace after the device-resident leg, so "
                              "its steps move a different number of experts over the link (expert_loads_per_step here "
                              "against h2d.loads_per_step) and, the step being link-bound, take proportionally long"}

    d, f = cfg.d_model, cfg.d_ff
    decode = cfg.name in ("mixtral_decode", "stack_decode", "dual_batch_stack")
    power_capped = bool(clocks and "sw_power_cap" in (clocks.get("reasons") or []))
    roofline = ffn_roofline(lg, kt, d, f, peaks, decode, "streaming step (a wave of hits + waves of misses, one launch per wave)",
                            gated=cfg.expert_kind == "swiglu", fill_peak=fill_peak, power_capped=power_capped)
    tr, stale, src = ncu_traffic(cfg.name, "in_step")
    roofline.update({"traffic": tr, "traffic_stale": stale, "traffic_source": src})
    res["roofline"] = roofline

    res["h2d"] = {"bytes_per_step": st["bytes_h2d"] / steps, "loads_per_step": (st["ondemand_loads"] + st["prefetch_issued"]) / steps,
                  "copy_busy_ms_per_step": copy_ms / steps,
                  "achieved_gbs": (st["bytes_h2d"] / (copy_ms * 1e-3) / 1e9) if copy_ms > 0 else None,
                  "peak_gbs": h2d_peak, "peak_source": "measured in this run on an idle device: pinned->device cudaMemcpyAsync, best of 10 over one "
                                 "expert-sized and one 1 GiB buffer",
                  "frac": (st["bytes_h2d"] / (copy_ms * 1e-3) / 1e9 / h2d_peak) if copy_ms > 0 and h2d_peak else None,
                  "gbs_over_step": st["bytes_h2d"] / (ms * 1e-3) / 1e9,
                  "step_ms_lower_bound_from_link": (st["bytes_h2d"] / steps / (h2d_peak * 1e9) * 1e3) if h2d_peak else None,
                  "copy_overlap": "copies run on the library's copy stream concurrently with the grouped-FFN waves"}
    res["cache"] = dict(st, hit_ratio=st["hits"] / max(1, st["lookups"]))
    res["phys"] = drv.phys or cfg.n_layers * cfg.n_experts

    counts = runner.counts.cpu().numpy()
    res["aux_roofline"] = aux_rooflines(runner, cfg, peaks, dev) if rank == 0 else None
    drv.close()
    if want_resident and rank == 0:
        res["roofline_resident"] = resident_leg(cfg, counts, peaks, dev, args, decode, fill_peak)
    return res


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
    fill_peak = measure_fill_peak(dev) if rank == 0 else None

    main = measure_workload(cfg, args, dev, plan, world, peaks, log, args.steps, args.warmup, want_e2e=True,
                            want_resident=not args.no_resident, fill_peak=fill_peak, local=local, rank=rank)

    # The default line also vouches for the other two north_star targets (BASELINE.json): decode expert-weight reads
    # against HBM (configs[2]) and the many-expert prefill GEMM against the tensor peak (configs[3]) -- short runs of
    # the same path on those workloads, each with its in-step and resident FFN roofline.
    extra = {}
    if args.workload == "mixtral_prefill" and world == 1 and not args.no_extra:
        for key, name, n_steps in (("decode", "mixtral_decode", 12), ("many_expert", "many_expert_prefill", 4)):
            c2 = wl.CONFIGS[name]
            p2 = replica_plan(rank, world, c2.T)
            r2 = measure_workload(c2, args, dev, p2, world, peaks, log, n_steps, 3, want_e2e=False, want_resident=True,
                                  fill_peak=fill_peak, local=local, rank=rank)
            extra[key] = {"config": workload_config(c2, world, {"phys_host_experts": r2["phys"], "cache_policy": args.policy}),
                          "steps": n_steps, "warmup": 3, "value": r2["value"], "unit": UNIT, "ms_per_step": r2["ms_per_step"],
                          "clocks": r2["clocks"], "gpu_launches": r2["gpu_launches"], "roofline": r2["roofline"],
                          "roofline_resident": r2.get("roofline_resident"), "h2d": r2["h2d"], "cache": r2["cache"],
                          "aux_roofline": r2["aux_roofline"]}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_baseline = cpu_baseline_block(cfg, args)

    if rank == 0:
        line = {"metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": main["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": workload_config(cfg, world, {"phys_host_experts": main["phys"], "cache_policy": args.policy}),
                "clocks": main["clocks"], "e2e": main["e2e"], "gpu_launches": main["gpu_launches"],
                "roofline": main["roofline"], "roofline_resident": main.get("roofline_resident"),
                "aux_roofline": main["aux_roofline"], "h2d": main["h2d"], "cache": main["cache"], "cpu_baseline": cpu_baseline}
        line.update(extra)
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
            runner.ctx.ef_get_kernel_times(reset=True); runner.ctx.ef_get_launch_log(reset=True)
            runner.ctx.ef_set_kernel_timing(True)
        l0 = runner.ctx.ef_launch_count()
        dist_barrier(); torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            step(sched, e2e)
        e1.record()
        runner.ctx.ef_sync(); torch.cuda.synchronize(); dist_barrier()
        ms = dist_max(e0.elapsed_time(e1), dev)
        kt = lg = None
        if with_kernel_times:
            kt = runner.ctx.ef_get_kernel_times(reset=True); lg = runner.ctx.ef_get_launch_log(reset=True)
            runner.ctx.ef_set_kernel_timing(False)
        st = runner.ctx.ef_cache_get_stats()
        copy_ms = runner.ctx.ef_copy_busy_ms()
        return {"ms": ms, "launches": runner.ctx.ef_launch_count() - l0, "kt": kt, "lg": lg, "st": st, "copy_ms": copy_ms}

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
    roofline = ffn_roofline(on["lg"], on["kt"], d, f, peaks, True, "streaming steps with the Token Scheduler on")
    st = on["st"]
    h2d = {"bytes_per_step": st["bytes_h2d"] / args.steps, "copy_busy_ms_per_step": on["copy_ms"] / args.steps,
           "achieved_gbs": st["bytes_h2d"] / (on["copy_ms"] * 1e-3) / 1e9 if on["copy_ms"] > 0 else None, "peak_gbs": h2d_peak,
           "frac": (st["bytes_h2d"] / (on["copy_ms"] * 1e-3) / 1e9 / h2d_peak) if on["copy_ms"] > 0 and h2d_peak else None}
    runner.close()
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_tok, n_lay = ref_sample_size(cfg, args)
        v, dt, cores, what = oracle_sample_dual(cfg, n_tok, n_lay)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what, "precision": "fp64"}
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


def ffn_roofline(lg, kt, d, f, peaks, decode, where, gated=True, fill_peak=None, power_capped=False, burst_only=False):
    """Roofline of the dominant kernel -- the grouped-FFN wave kernel (both GEMMs of a wave in one launch; a wave whose
    expert is still arriving in two chunks runs them as two launches) -- from the library's per-launch CUDA events.
    lg: the launch log (ef_get_launch_log), kt: the totals (ef_get_kernel_times).
    Algorithmic work of a launch over `rows` routed rows in `groups` experts (gated = SwiGLU experts):
      GEMM1  (4 | 2) d f FLOP per row, (4 | 2) d f weight bytes per expert, 2 d read + 2 f written per row
      GEMM2        2 d f FLOP per row,       2 d f weight bytes per expert, 2 f read + 2 d written per row
    `frac` holds the whole path against ONE roofline (tensor peak for prefill, HBM for decode); `frac_of_launch_bound`
    holds every launch against ITS OWN bound max(FLOP / tensor peak, bytes / HBM bandwidth), which is the honest figure
    for waves of a few small experts that no tensor pipe could keep busy (their weights have to come out of HBM once)."""
    g1 = 4.0 if gated else 2.0
    burst, sust, hbm = peaks["bf16_tflops"], peaks.get("bf16_tflops_sustained") or peaks["bf16_tflops"], peaks["hbm_gbs"]
    tot = {"t": 0.0, "flop": 0.0, "wbytes": 0.0, "bytes": 0.0, "bound_burst": 0.0, "bound_sust": 0.0}
    kinds = {1: dict(t=0.0, n=0, flop=0.0, wbytes=0.0), 2: dict(t=0.0, n=0, flop=0.0, wbytes=0.0), 3: dict(t=0.0, n=0, flop=0.0, wbytes=0.0)}
    for r in lg:
        w1, w2 = (1 if r["which"] & 1 else 0), (1 if r["which"] & 2 else 0)
        flop = (w1 * g1 + w2 * 2.0) * d * f * r["rows"]
        wb = (w1 * g1 + w2 * 2.0) * d * f * r["groups"]
        ab = (w1 + w2) * (2.0 * d + 2.0 * f) * r["rows"]
        t = r["ms"] * 1e-3
        tot["t"] += t; tot["flop"] += flop; tot["wbytes"] += wb; tot["bytes"] += wb + ab
        tot["bound_burst"] += max(flop / (burst * 1e12), (wb + ab) / (hbm * 1e9))
        tot["bound_sust"] += max(flop / (sust * 1e12), (wb + ab) / (hbm * 1e9))
        k = kinds[r["which"]]
        k["t"] += t; k["n"] += 1; k["flop"] += flop; k["wbytes"] += wb
    T = max(tot["t"], 1e-12)
    n = max(1, len(lg))

    def kind_view(k):
        if not k["n"]:
            return None
        v = {"launches": k["n"], "avg_launch_ms": k["t"] * 1e3 / k["n"], "tflops": k["flop"] / k["t"] / 1e12,
             "weight_gbs": k["wbytes"] / k["t"] / 1e9}
        v["frac"] = v["weight_gbs"] / hbm if decode else v["tflops"] / burst
        return v
    out = {"kernel": f"ffn_wave_kernel (tcgen05 grouped GEMM1 + GEMM2 of a wave, one launch), {where}",
           "launches": len(lg), "avg_launch_ms": tot["t"] * 1e3 / n, "rows_per_launch": sum(r["rows"] for r in lg) / n,
           "groups_per_launch": sum(r["groups"] for r in lg) / n,
           "algorithmic_bytes_per_launch": tot["bytes"] / n, "algorithmic_flop_per_launch": tot["flop"] / n,
           "frac_of_launch_bound": tot["bound_burst"] / T,
           "frac_of_launch_bound_note": "sum over launches of max(FLOP / burst bf16 peak, algorithmic bytes / HBM copy bandwidth) "
                                        "divided by the sum of their measured durations",
           "by_launch_kind": {"wave (GEMM1+GEMM2, one launch)": kind_view(kinds[3]), "gemm1 only": kind_view(kinds[1]),
                              "gemm2 only": kind_view(kinds[2])}}
    if decode:
        a = tot["wbytes"] / T / 1e9
        out.update({"bound": "hbm", "achieved": a, "peak": hbm, "unit": "GB/s", "frac": a / hbm,
                    "peak_source": f"{peaks['source']} HBM copy bandwidth (read + write; a read-only stream measures higher)"})
    else:
        a = tot["flop"] / T / 1e12
        # a link-bound step leaves the GPU idle most of the time: its kernels run at burst clocks unless the sampled
        # clocks say the power cap was active; the resident leg is always a kernel timed alone (burst)
        use_burst = burst_only or not power_capped
        out.update({"bound": "tensor", "achieved": a, "peak": burst if use_burst else sust, "unit": "TFLOP/s",
                    "frac": a / (burst if use_burst else sust), "frac_burst": a / burst, "frac_sustained": a / sust,
                    "peak_source": f"{peaks['source']} bf16 " + ("burst (kernel timed alone, or inside a step whose sampled clocks "
                                   "show no power cap)" if use_burst else "sustained (power cap active in the sampled clocks)")})
        if fill_peak and kt and kt.get("gemm1_fill_bytes"):
            fb = kt["gemm1_fill_bytes"] + kt["gemm2_fill_bytes"]
            out["l2_to_sm"] = {"bound": "l2_to_sm", "achieved": fb / T / 1e9, "peak": fill_peak, "unit": "GB/s",
                               "frac": fb / T / 1e9 / fill_peak, "bytes_per_launch": fb / n, "flop_per_fill_byte": tot["flop"] / fb,
                               "peak_source": "measured in this run by the diagnostic library's probe (ef_diag_tma_fill_gbs): every "
                                              "SM streaming 32 KB TMA boxes out of a 64 MB L2-resident region"}
    return out


def resident_leg(cfg, counts, peaks, dev, args, decode, fill_peak=None):
    """The grouped FFN alone with every active expert of one visit resident (kernel-only roofline): ONE launch over all
    groups running both GEMMs, timed by the library's CUDA events on the compute stream, weights > L2 or L2 flushed."""
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
    # when the active experts' weights could stay in L2 between launches, flush it
    flush = None
    if len(act) * cfg.expert_bytes < 512e6:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ctx.ef_sync()
    for _ in range(3):
        ctx.ef_expert_ffn_grouped_resident(x_perm, rb, rw, sl, y)
    ctx.ef_sync()
    ctx.ef_set_kernel_timing(True)
    ctx.ef_get_kernel_times(reset=True); ctx.ef_get_launch_log(reset=True)
    n = max(5, args.steps)
    for _ in range(n):
        if flush is not None:
            flush.zero_()
        ctx.ef_expert_ffn_grouped_resident(x_perm, rb, rw, sl, y)
    kt = ctx.ef_get_kernel_times(reset=True)
    lg = ctx.ef_get_launch_log(reset=True)
    res = ffn_roofline(lg, kt, cfg.d_model, cfg.d_ff, peaks, decode,
                       "all active experts of one visit resident, one launch over all groups",
                       gated=cfg.expert_kind == "swiglu", fill_peak=fill_peak, burst_only=True)
    tr, stale, src = ncu_traffic(cfg.name, "resident")
    res.update({"traffic": tr, "traffic_stale": stale, "traffic_source": src})
    res["rows_per_expert"] = [int(c) for c in counts]
    res["l2"] = "256 MB flush write between launches" if flush is not None else "weights exceed L2 between launches"
    ctx.close()
    return res


def aux_rooflines(runner, cfg, peaks, dev):
    """HBM rooflines of the memory-bound kernels of the path (S 8(d): route, permute = index + gather, combine, rmsnorm):
    algorithmic bytes per call / CUDA-event time per call / measured HBM copy bandwidth.  Each kernel is timed over back to
    back calls that rotate through enough input / output buffer sets to exceed L2 (so no call re-reads what the previous
    one left there), after a warm-up; the buffers are scratch copies, the runner's own state is not touched."""
    import torch
    T, d, k, E = cfg.T, cfg.d_model, cfg.top_k, cfg.n_experts
    R = T * k
    c = runner.ctx
    hbm = peaks["hbm_gbs"]
    per_set = max(1, R * d * 2 + T * d * 2)
    n_sets = int(min(64, max(2, (300 << 20) // per_set + 1)))
    bf = torch.bfloat16
    xs = [torch.randn((T, d), device=dev, dtype=torch.float32).to(bf) for _ in range(n_sets)]
    xps = [torch.empty((R, d), dtype=bf, device=dev) for _ in range(n_sets)]
    outs = [torch.empty((T, d), dtype=bf, device=dev) for _ in range(n_sets)]
    layer = 0
    wr, bias = runner.w_router[layer], runner.bias[layer]
    idx = torch.empty((T, k), dtype=torch.int32, device=dev); w = torch.empty((T, k), dtype=torch.float32, device=dev)
    counts = torch.empty((E,), dtype=torch.int32, device=dev); offsets = torch.empty((E + 1,), dtype=torch.int32, device=dev)
    src = torch.empty((R,), dtype=torch.int32, device=dev); inv = torch.empty((R,), dtype=torch.int32, device=dev)
    c.ef_route_topk(xs[0], wr, bias, T, cfg.renorm, idx, w, None)
    c.ef_permute(idx, xs[0], T, xps[0], counts, offsets, src, inv)
    torch.cuda.synchronize()
    reps = 3 * n_sets
    cap_stream = torch.cuda.Stream(device=dev)

    def timed(fn):
        # the calls are captured into ONE CUDA graph and the graph is replayed: per-call time = kernel time + the gap
        # between two graph nodes, without the ~10 us a ctypes call from Python costs on the host
        for i in range(n_sets):
            fn(i)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=cap_stream):
            for i in range(reps):
                fn(i % n_sets)
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        g.replay()
        e1.record(); e1.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / reps
    rows = {}

    def add(name, secs, nbytes, what):
        rows[name] = {"bound": "hbm", "us_per_call": secs * 1e6, "algorithmic_bytes": nbytes, "achieved": nbytes / secs / 1e9,
                      "peak": hbm, "unit": "GB/s", "frac": nbytes / secs / 1e9 / hbm, "bytes": what}
    add("route_topk", timed(lambda i: c.ef_route_topk(xs[i], wr, bias, T, cfg.renorm, idx, w, None)),
        T * d * 2 + E * d * 2 + T * k * 8, "x [T,d] bf16 + router [E,d] bf16 read, idx + w [T,k] written")
    add("permute (index + gather)", timed(lambda i: c.ef_permute(idx, xs[i], T, xps[i], counts, offsets, src, inv)),
        T * d * 2 + R * d * 2 + R * 12, "x [T,d] read once (k-fold re-read from L2), x_perm [R,d] written, idx read + src + inv written")
    add("combine", timed(lambda i: c.ef_combine(xps[i], inv, w, T, None, None, outs[i])),
        R * d * 2 + T * d * 2 + R * 8, "y_perm [R,d] read, out [T,d] written, inv + w read")
    if cfg.n_layers > 1:
        add("rmsnorm", timed(lambda i: c.ef_rmsnorm(xs[i], T, 1e-5, outs[i])), 2 * T * d * 2, "x [T,d] read, out [T,d] written")
    return {"kernels": rows, "peak_source": f"{peaks['source']} HBM copy bandwidth",
            "how": f"CUDA events around the replay of one CUDA graph holding {reps} calls that rotate through {n_sets} buffer "
                   f"sets ({n_sets * per_set / 1e6:.0f} MB > L2), after {n_sets} eager warm-up calls and one warm-up replay"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="mixtral_prefill", choices=sorted(wl.CONFIGS))
    ap.add_argument("--ref-tokens", type=int, default=0, help="tokens in the bounded oracle sample (0 = per-workload default)")
    ap.add_argument("--ref-layers", type=int, default=0, help="layer visits in the bounded oracle sample (0 = default)")
    ap.add_argument("--ref-precision", default="fp64", choices=["fp64", "fp32"],
                    help="--impl reference: the oracle as the parity tests use it (fp64) or the same C file built with "
                         "-DORC_REAL=float")
    ap.add_argument("--phys-experts", type=int, default=0,
                    help="alias the logical experts onto this many physical pinned host buffers (0 = one per expert "
                         "if host memory allows)")
    ap.add_argument("--horizon", type=int, default=None,
                    help="override the workload's prefetch horizon H in visits (<= 0: as far as the supplied path reaches; R10)")
    ap.add_argument("--no-early-release", action="store_true",
                    help="EF_OPT_EARLY_RELEASE = 0: the first-victim hit always runs as a wave of its own (A/B arm)")
    ap.add_argument("--policy", default="plec", choices=["plec", "lru", "layer_lru", "next_layer_all"],
                    help="cache policy arm: the paper's PLEC (default), on-demand LRU over the pool, LRU inside a per-layer "
                         "share, or PLEC prefetching every expert of the next layer (the baselines of P:L230 as policy sketches)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-resident", action="store_true")
    ap.add_argument("--no-extra", action="store_true",
                    help="default workload only: skip the decode / many_expert blocks (the other two north_star targets)")
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
