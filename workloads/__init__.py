"""Seeded synthetic inputs for the ExpertFlow MoE-layer hot path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2410_17954_b200/``).  It holds none of the method's arithmetic: no
router, no top-k, no FFN, no cache policy.  It only draws random numbers
(numpy Philox, a counter-based generator keyed by ``(seed, tensor name, chunk)``),
rounds normals to bf16 bit patterns, and samples the *structure* of the paper's
workloads (expert-popularity skew, temporal locality, cross-layer locality,
imperfect predicted routing paths).  The recipe per configuration is stated in
DESIGN.md §5 and follows SURVEY.md §8(d) / BASELINE.json ``configs``.

The paper's datasets (WMT16, XSUM) and model weights are not
available; these inputs take their shapes and statistics only.

All tensors are numpy arrays; bf16 tensors are ``uint16`` bit patterns.
"""
from __future__ import annotations

import zlib
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np

_CHUNK = 1 << 22  # elements per independently keyed Philox stream


# ----------------------------------------------------------------------------
# bf16 <-> fp32 bit conversions (storage format only)
# ----------------------------------------------------------------------------
def f32_to_bf16_bits(a: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns."""
    u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)
    r = (u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns to fp32."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


# ----------------------------------------------------------------------------
# keyed random streams
# ----------------------------------------------------------------------------
def _key(seed: int, name: str, chunk: int = 0) -> list[int]:
    h = zlib.crc32(name.encode()) & 0xFFFFFFFF
    return [(int(seed) & 0xFFFFFFFF) | (h << 32), int(chunk)]


def stream(seed: int, name: str, chunk: int = 0) -> np.random.Generator:
    """A Philox generator keyed by (seed, tensor name, chunk): every tensor is
    reproducible on its own, independent of generation order."""
    return np.random.Generator(np.random.Philox(key=_key(seed, name, chunk)))


def normal_f32(seed: int, name: str, shape, std: float, threads: int = 8) -> np.ndarray:
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.float32)

    def fill(c):
        lo = c * _CHUNK
        hi = min(n, lo + _CHUNK)
        g = stream(seed, name, c)
        g.standard_normal(hi - lo, dtype=np.float32, out=out[lo:hi])
        out[lo:hi] *= np.float32(std)

    nchunks = (n + _CHUNK - 1) // _CHUNK
    if nchunks <= 1 or threads <= 1:
        for c in range(nchunks):
            fill(c)
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(fill, range(nchunks)))
    return out.reshape(shape)


def normal_bf16(seed: int, name: str, shape, std: float, threads: int = 8) -> np.ndarray:
    """N(0, std) rounded to bf16 (RNE); uint16 bit patterns."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.uint16)

    def fill(c):
        lo = c * _CHUNK
        hi = min(n, lo + _CHUNK)
        g = stream(seed, name, c)
        a = g.standard_normal(hi - lo, dtype=np.float32)
        a *= np.float32(std)
        out[lo:hi] = f32_to_bf16_bits(a)

    nchunks = (n + _CHUNK - 1) // _CHUNK
    if nchunks <= 1 or threads <= 1:
        for c in range(nchunks):
            fill(c)
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(fill, range(nchunks)))
    return out.reshape(shape)


# ----------------------------------------------------------------------------
# configurations (BASELINE.json "configs", SURVEY.md §8 size table)
# ----------------------------------------------------------------------------
@dataclass(frozen=True)
class MoEConfig:
    name: str
    T: int                 # tokens per visit
    d_model: int
    d_ff: int
    n_experts: int         # routed experts per layer
    top_k: int
    n_slots: int           # cache slots (global pool)
    n_layers: int = 1
    n_shared: int = 0      # always-resident shared experts per layer
    n_steps: int = 1       # decode steps (a step = n_layers visits)
    seed: int = 0
    w_std: float = 0.02
    renorm: int = 1
    # routing structure
    bias_kind: str = "none"    # none | normal | zipf | trace
    bias_std: float = 0.5
    zipf_s: float = 1.1
    keep_prob: float = 0.0     # temporal locality (cfg 3)
    layer_corr: float = 0.0    # cross-layer locality (cfg 5)
    pred_acc: float = 1.0      # token-level predictor accuracy
    horizon: int = 0           # prefetch horizon in visits; <=0 = fill
    trace_margin: float = 12.0
    phys_experts: int = 0      # >0: alias logical experts onto this many physical host buffers
    expert_kind: str = "swiglu"  # swiglu (BASELINE.json) | relu: Switch-style non-gated FFN (R30)

    @property
    def R(self) -> int:
        return self.T * self.top_k

    @property
    def expert_bytes(self) -> int:
        return (3 if self.expert_kind == "swiglu" else 2) * self.d_model * self.d_ff * 2

    @property
    def n_visits(self) -> int:
        return self.n_steps * self.n_layers


CONFIGS = {
    # cfg 1: tiny (BASELINE.json configs[0])
    "tiny": MoEConfig("tiny", T=64, d_model=256, d_ff=512, n_experts=8, top_k=2, n_slots=4, seed=0),
    # cfg 2: Mixtral-8x7B-shaped prefill (configs[1]) -- the headline config
    "mixtral_prefill": MoEConfig("mixtral_prefill", T=2048, d_model=4096, d_ff=14336, n_experts=8, top_k=2,
                                 n_slots=4, seed=2, bias_kind="normal", bias_std=0.5),
    # cfg 3: Mixtral-shaped decode, 16 tokens/step x 256 steps (configs[2])
    "mixtral_decode": MoEConfig("mixtral_decode", T=16, d_model=4096, d_ff=14336, n_experts=8, top_k=2,
                                n_slots=6, n_steps=256, seed=3, bias_kind="trace", keep_prob=0.6,
                                pred_acc=0.85, horizon=1),
    # cfg 4: many-expert prefill with 2 shared experts (configs[3])
    "many_expert_prefill": MoEConfig("many_expert_prefill", T=4096, d_model=2048, d_ff=1408, n_experts=64,
                                     top_k=6, n_slots=24, n_shared=2, seed=4, bias_kind="zipf", zipf_s=1.1),
    # cfg 5: 32-layer Mixtral-shaped stack decode (configs[4])
    "stack_decode": MoEConfig("stack_decode", T=64, d_model=4096, d_ff=14336, n_experts=8, top_k=2,
                              n_slots=64, n_layers=32, n_steps=128, seed=5, bias_kind="trace",
                              layer_corr=0.5, pred_acc=0.8, horizon=0),
    # f4: Switch-style layer (the paper's own model family: Switch-32/64/128): top-1, gate weight = full
    # softmax probability (Eq. 2, renorm=0), non-gated ReLU experts of Switch-base size, cache of 16 of 64 experts
    "switch_prefill": MoEConfig("switch_prefill", T=4096, d_model=768, d_ff=3072, n_experts=64, top_k=1, n_slots=16,
                                seed=7, renorm=0, bias_kind="zipf", zipf_s=1.1, expert_kind="relu"),
    # f1: the cfg 5 stack fed by TWO incoming batches of 16 decode tokens per step, rebatched by the Token Scheduler
    # (PAPER.md 3.3 / 4.2); same shapes, cache and predictor accuracy as cfg 5
    "dual_batch_stack": MoEConfig("dual_batch_stack", T=16, d_model=4096, d_ff=14336, n_experts=8, top_k=2,
                                  n_slots=64, n_layers=32, n_steps=64, seed=6, bias_kind="trace",
                                  pred_acc=0.8, horizon=0),
}


def scaled(cfg: MoEConfig, **kw) -> MoEConfig:
    """A copy of cfg with some fields replaced (used for reduced-size parity cases)."""
    d = {f: getattr(cfg, f) for f in cfg.__dataclass_fields__}
    d.update(kw)
    return MoEConfig(**d)


# ----------------------------------------------------------------------------
# tensors
# ----------------------------------------------------------------------------
def activations(cfg: MoEConfig, step: int = 0) -> np.ndarray:
    """x[T, d] bf16 ~ N(0,1); a fresh draw per decode step."""
    return normal_bf16(cfg.seed, f"x.step{step}", (cfg.T, cfg.d_model), 1.0)


def router_weight(cfg: MoEConfig, layer: int = 0) -> np.ndarray:
    """Wr[E, d] bf16 ~ N(0, 1/sqrt(d)) so that x.Wr ~ N(0,1)."""
    return normal_bf16(cfg.seed, f"wr.l{layer}", (cfg.n_experts, cfg.d_model), 1.0 / np.sqrt(cfg.d_model))


def expert_weights(cfg: MoEConfig, layer: int, expert: int, threads: int = 8):
    """(Wg[f,d], Wu[f,d], Wd[d,f]) bf16 ~ N(0, w_std).  expert < 0 names shared expert (-1 - s).
    With cfg.phys_experts > 0 logical experts alias onto that many physical draws."""
    gid = layer * cfg.n_experts + expert if expert >= 0 else None
    if gid is not None and cfg.phys_experts > 0:
        tag = f"phys{gid % cfg.phys_experts}"
    elif gid is not None:
        tag = f"l{layer}.e{expert}"
    else:
        tag = f"l{layer}.shared{-1 - expert}"
    f, d = cfg.d_ff, cfg.d_model
    wg = normal_bf16(cfg.seed, f"wg.{tag}", (f, d), cfg.w_std, threads)
    wu = normal_bf16(cfg.seed, f"wu.{tag}", (f, d), cfg.w_std, threads) if cfg.expert_kind == "swiglu" else None
    wd = normal_bf16(cfg.seed, f"wd.{tag}", (d, f), cfg.w_std, threads)
    return wg, wu, wd


def static_router_bias(cfg: MoEConfig, layer: int = 0) -> np.ndarray | None:
    """Per-expert fp32 bias [E] producing popularity skew (cfg 2: N(0,0.5); cfg 4: Zipf)."""
    E = cfg.n_experts
    if cfg.bias_kind == "normal":
        return normal_f32(cfg.seed, f"bias.l{layer}", (E,), cfg.bias_std)
    if cfg.bias_kind == "zipf":
        # popularity p_e ~ rank^-s  <=>  additive logit bias -s*ln(rank); rank order is a seeded permutation
        rank = stream(cfg.seed, f"zipfperm.l{layer}").permutation(E) + 1
        return (-cfg.zipf_s * np.log(rank.astype(np.float64))).astype(np.float32)
    return None


# ----------------------------------------------------------------------------
# routing traces (cfg 3, cfg 5) and predicted paths
# ----------------------------------------------------------------------------
@dataclass
class Trace:
    """Intended routing of a decode run.  sets[v][t] is the ordered k-tuple of experts
    token-slot t is driven to at visit v (first = highest logit)."""
    sets: np.ndarray            # int32 [n_visits, T, k]
    predicted: np.ndarray       # uint8 [n_visits, E]  batch-level predicted path (OR over tokens)
    actual: np.ndarray          # uint8 [n_visits, E]  batch-level intended path
    meta: dict = field(default_factory=dict)


def _draw_set(g: np.random.Generator, p: np.ndarray, k: int) -> np.ndarray:
    return g.choice(p.shape[0], size=k, replace=False, p=p).astype(np.int32)


def routing_trace(cfg: MoEConfig, n_steps: int | None = None) -> Trace:
    """Sample per-token expert sets with temporal locality (keep_prob: a sequence slot keeps
    its previous step's set in the same layer, PAPER L245 'TLP') and cross-layer locality
    (layer_corr: reuse the set of the layer below, same local ids, PAPER L245 'SLP'), then a
    predicted path: per token, with prob pred_acc the predicted set equals the intended set,
    else a uniform random k-subset; batch-level path = OR over tokens."""
    n_steps = cfg.n_steps if n_steps is None else n_steps
    L, T, k, E = cfg.n_layers, cfg.T, cfg.top_k, cfg.n_experts
    g = stream(cfg.seed, "trace")
    # per-layer expert popularity: softmax of N(0,1) offsets
    pops = []
    for l in range(L):
        o = stream(cfg.seed, f"traceoff.l{l}").standard_normal(E)
        p = np.exp(o - o.max())
        pops.append(p / p.sum())
    nv = n_steps * L
    sets = np.zeros((nv, T, k), dtype=np.int32)
    for s in range(n_steps):
        for l in range(L):
            v = s * L + l
            for t in range(T):
                u = g.random()
                if l > 0 and u < cfg.layer_corr:
                    sets[v, t] = sets[v - 1, t]
                elif s > 0 and g.random() < cfg.keep_prob:
                    sets[v, t] = sets[v - L, t]
                else:
                    sets[v, t] = _draw_set(g, pops[l], k)
    gp = stream(cfg.seed, "trace.pred")
    predicted = np.zeros((nv, E), dtype=np.uint8)
    actual = np.zeros((nv, E), dtype=np.uint8)
    for v in range(nv):
        for t in range(T):
            actual[v, sets[v, t]] = 1
            if gp.random() < cfg.pred_acc:
                predicted[v, sets[v, t]] = 1
            else:
                predicted[v, gp.choice(E, size=k, replace=False)] = 1
    return Trace(sets=sets, predicted=predicted, actual=actual, meta={"L": L, "T": T, "k": k, "E": E})


def trace_bias(cfg: MoEConfig, trace: Trace, visit: int) -> np.ndarray:
    """Per-token fp32 bias [T, E] that drives the router to trace.sets[visit]: the j-th intended
    expert gets +margin + (k-1-j), everything else 0.  The margin (default 12) dominates the
    natural logits x.Wr ~ N(0,1), so routing does not depend on activation round-off."""
    T, k, E = cfg.T, cfg.top_k, cfg.n_experts
    b = np.zeros((T, E), dtype=np.float32)
    for j in range(k):
        b[np.arange(T), trace.sets[visit, :, j]] = np.float32(cfg.trace_margin + (k - 1 - j))
    return b


# ----------------------------------------------------------------------------
# token-level routing paths for the Token Scheduler (§3.3)
# ----------------------------------------------------------------------------
def token_paths(seed: int, n_tokens: int, n_layers: int, n_experts: int, top_k: int, n_families: int = 2,
                family_prob: float = 0.8) -> np.ndarray:
    """Binary routing-path matrices r[N, L, E] (uint8 0/1, exactly top_k ones per layer) with the structure
    the Token Scheduler exploits: every token belongs to one of n_families latent groups ("tokens sharing similar
    routing paths"); per layer a token takes its family's expert set with probability family_prob, else a
    fresh top_k draw from that layer's popularity (softmax of N(0,1) offsets, as in routing_trace).  Families are
    interleaved at random over the token index, so the incoming batches [0, T) and [T, 2T) mix them."""
    g = stream(seed, f"tokpaths.N{n_tokens}.L{n_layers}.E{n_experts}.k{top_k}.F{n_families}")
    pops = []
    for l in range(n_layers):
        o = g.standard_normal(n_experts)
        p = np.exp(o - o.max())
        pops.append(p / p.sum())
    fam_sets = np.zeros((n_families, n_layers, top_k), np.int64)
    for f in range(n_families):
        for l in range(n_layers):
            fam_sets[f, l] = _draw_set(g, pops[l], top_k)
    fam = g.integers(0, n_families, size=n_tokens)
    r = np.zeros((n_tokens, n_layers, n_experts), np.uint8)
    for i in range(n_tokens):
        for l in range(n_layers):
            es = fam_sets[fam[i], l] if g.random() < family_prob else _draw_set(g, pops[l], top_k)
            r[i, l, es] = 1
    return r


# ----------------------------------------------------------------------------
# dual-batch decode traces (Token Scheduler end to end; §3.3, §4.2)
# ----------------------------------------------------------------------------
@dataclass
class DualBatchTrace:
    """Two incoming batches of cfg.T tokens per step (global token index i < N = 2T: batch i // T).
    sets[s, i, l] is the ordered k-tuple of experts token i is driven to in layer l at step s; pred_sets is the
    routing-path predictor's output for the same token (R17: equal to sets with prob pred_acc, else a uniform
    random k-subset, drawn per token and layer)."""
    sets: np.ndarray         # int32 [n_steps, N, L, k]
    pred_sets: np.ndarray    # int32 [n_steps, N, L, k]
    family: np.ndarray       # int32 [N] latent group of every sequence slot (kept over the steps)


def dual_batch_trace(cfg: MoEConfig, n_steps: int, n_families: int = 2, family_prob: float = 0.8) -> DualBatchTrace:
    """Sequence slots belong to latent families ("tokens sharing similar routing paths") that are mixed at
    random over the two incoming batches.  Per step and layer a token takes its family's expert set with
    probability family_prob, else a fresh draw from the layer's popularity."""
    L, T, k, E = cfg.n_layers, cfg.T, cfg.top_k, cfg.n_experts
    N = 2 * T
    g = stream(cfg.seed, f"dualtrace.F{n_families}")
    pops = []
    for l in range(L):
        o = g.standard_normal(E)
        p = np.exp(o - o.max())
        pops.append(p / p.sum())
    fam_sets = np.zeros((n_families, L, k), np.int32)
    for f in range(n_families):
        for l in range(L):
            fam_sets[f, l] = _draw_set(g, pops[l], k)
    family = g.integers(0, n_families, size=N).astype(np.int32)
    sets = np.zeros((n_steps, N, L, k), np.int32)
    pred = np.zeros_like(sets)
    for s in range(n_steps):
        for i in range(N):
            for l in range(L):
                sets[s, i, l] = fam_sets[family[i], l] if g.random() < family_prob else _draw_set(g, pops[l], k)
                pred[s, i, l] = sets[s, i, l] if g.random() < cfg.pred_acc else g.choice(E, size=k, replace=False)
    return DualBatchTrace(sets=sets, pred_sets=pred, family=family)


def sets_to_paths(sets: np.ndarray, n_experts: int) -> np.ndarray:
    """[N, L, k] expert ids -> binary routing-path matrices uint8 [N, L, E]."""
    N, L, _ = sets.shape
    r = np.zeros((N, L, n_experts), np.uint8)
    r[np.arange(N)[:, None, None], np.arange(L)[None, :, None], sets] = 1
    return r


def bias_from_sets(cfg: MoEConfig, sets: np.ndarray) -> np.ndarray:
    """fp32 [N, L, E] router bias that drives token i in layer l to sets[i, l] in order (as trace_bias does)."""
    N, L, k = sets.shape
    b = np.zeros((N, L, cfg.n_experts), np.float32)
    for j in range(k):
        b[np.arange(N)[:, None], np.arange(L)[None, :], sets[:, :, j]] = np.float32(cfg.trace_margin + (k - 1 - j))
    return b
