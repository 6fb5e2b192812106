"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (MoELayerRunner.visit with
the configured number of cache slots, so experts stream in waves), checked on what the oracle can afford:

* integers (top-k on the GPU's own logits, counts, offsets, permutation, slot table, cache counters): bit-exact,
  over the whole tensors;
* float outputs: a seeded sample of tokens, each computed by the oracle one by one (route -> FFN of its k experts
  -> combine [-> 32-layer chain for cfg 5]) and compared under the north_star tolerance.
"""
import numpy as np
import pytest

import oracle
import workloads as wl
from oracle.cache_sim import CacheSim, STAT_KEYS

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from test_gpu_stages import bf, check_float, dev_bf16, to_bits  # noqa: E402


def make_runner(cfg, experts, horizon=None):
    """experts: dict (layer, e) -> (wg, wu, wd); entries that are the same object are registered once and aliased."""
    from paper_2410_17954_b200 import MoELayerRunner
    r = MoELayerRunner(cfg.n_layers, cfg.n_experts, cfg.top_k, cfg.d_model, cfg.d_ff, cfg.n_slots, cfg.n_shared,
                       cfg.T, cfg.horizon if horizon is None else horizon, cfg.renorm)
    first = {}
    for l in range(cfg.n_layers):
        r.set_router(l, wl.router_weight(cfg, l), wl.static_router_bias(cfg, l))
        for e in range(cfg.n_experts):
            w3 = experts[(l, e)]
            if id(w3) in first:
                r.ctx.ef_host_expert_alias(l, e, *first[id(w3)])
            else:
                r.register_expert(l, e, *w3)
                first[id(w3)] = (l, e)
        for s in range(cfg.n_shared):
            r.register_expert(l, -1 - s, *experts[(l, -1 - s)])
    return r


def assert_cache_equal(runner, sim):
    assert runner.ctx.ef_cache_snapshot() == sim.snapshot()
    st = runner.ctx.ef_cache_get_stats()
    assert st == {k: sim.stats[k] for k in STAT_KEYS}


def check_integers(r, x, wr, bias, cfg):
    """Top-k from the GPU's own logits (R22), then counts / offsets / permutation bit-exact."""
    logits_gpu = r.logits[:cfg.T].cpu().numpy()
    ref_logits = oracle.router_logits(x, wr, bias)
    np.testing.assert_allclose(logits_gpu, ref_logits, rtol=0, atol=2e-3)
    idx_ref, w_ref = oracle.topk_gate(logits_gpu.astype(np.float64), cfg.top_k, cfg.renorm)
    assert np.array_equal(r.topk_idx[:cfg.T].cpu().numpy(), idx_ref)
    np.testing.assert_allclose(r.topk_w[:cfg.T].cpu().numpy(), w_ref, rtol=2e-4)
    counts, offsets, src, inv = oracle.permute(idx_ref, cfg.n_experts)
    assert np.array_equal(r.counts.cpu().numpy(), counts)
    assert np.array_equal(r.offsets.cpu().numpy(), offsets)
    assert np.array_equal(r.src[:cfg.R].cpu().numpy(), src)
    assert np.array_equal(r.inv[:cfg.R].cpu().numpy(), inv)
    assert np.array_equal(to_bits(r.x_perm[:cfg.R]), oracle.gather_rows(x, src, cfg.top_k))
    return idx_ref, counts


def prefill_case(name, n_sample, steps):
    cfg = wl.CONFIGS[name]
    ex = {(0, e): wl.expert_weights(cfg, 0, e, threads=16) for e in range(cfg.n_experts)}
    for s in range(cfg.n_shared):
        ex[(0, -1 - s)] = wl.expert_weights(cfg, 0, -1 - s)
    r = make_runner(cfg, ex)
    x = wl.activations(cfg)
    wr, bias = wl.router_weight(cfg), wl.static_router_bias(cfg)
    sim = CacheSim(1, cfg.n_experts, cfg.n_slots, cfg.expert_bytes, cfg.horizon)
    ones = np.ones((1, cfg.n_experts), np.uint8)
    sim.prefetch(-1, ones); r.ctx.ef_cache_prefetch(-1, ones)
    xd = dev_bf16(x)
    out = torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16, device="cuda")
    rows = np.sort(wl.stream(cfg.seed, "fullsize.sample").choice(cfg.T, size=n_sample, replace=False))
    ref = None
    for v in range(steps):                 # the same batch every step, cache state carried over (as bench.py does)
        out.zero_()
        r.visit(v, xd, out, predicted_next=ones, want_logits=True)
        r.ctx.ef_sync()
        idx_ref, counts = check_integers(r, x, wr, bias, cfg)
        sim.visit(v, counts); sim.prefetch(v, ones)
        assert_cache_equal(r, sim)
        if ref is None:
            ref = oracle.layer_forward(x, wr, bias, lambda e: ex[(0, e)], cfg.top_k, cfg.renorm,
                                       shared=[ex[(0, -1 - s)] for s in range(cfg.n_shared)], rows=rows)
            assert np.array_equal(ref.idx, idx_ref)          # routing margin holds at this draw (R22)
        check_float(bf(to_bits(out))[rows], ref.out)
    st = r.ctx.ef_cache_get_stats()
    r.close()
    return cfg, st, counts


def test_cfg2_mixtral_prefill_full_size():
    cfg, st, counts = prefill_case("mixtral_prefill", n_sample=48, steps=2)
    assert counts.sum() == cfg.T * cfg.top_k and (counts > 0).all()
    # 4 slots, 8 active experts: warm-up prefetch of 4, then 4 on-demand loads in step 0 and 4 in step 1
    assert st["prefetch_issued"] == 4 and st["ondemand_loads"] == 8 and st["hits"] == 8
    assert st["bytes_h2d"] == 12 * cfg.expert_bytes


def test_cfg4_many_expert_prefill_full_size():
    cfg, st, counts = prefill_case("many_expert_prefill", n_sample=96, steps=2)
    assert counts.sum() == cfg.T * cfg.top_k
    assert st["misses"] >= 2 * (int((counts > 0).sum()) - cfg.n_slots)


def decode_case(cfg, n_steps, sample_tokens, phys=0, forced_tokens=()):
    """Full-shape decode trace: accounting bit-exact at every visit; float outputs of sampled tokens against the
    oracle's own per-token chain (route -> FFN of its k experts -> combine, layer after layer; nothing flows from the
    GPU into the oracle).
      * `forced_tokens` (stacks only): before each visit the GPU's rows for these tokens are overwritten with the
        ORACLE's bf16 layer input, so every layer is compared on identical inputs under the per-layer north_star
        tolerance (teacher forcing from the oracle side, as in test_gpu_stages.py);
      * `sample_tokens` run free on the GPU through all L layers; their error against the oracle's own chain is
        measured after every layer and returned (free_err: mean relative, free_max: max abs / max|ref|) -- the caller
        asserts on the measurement."""
    L, E, k = cfg.n_layers, cfg.n_experts, cfg.top_k
    n_phys = phys if phys else L * E
    gen = wl.scaled(cfg, phys_experts=phys)
    store = {}
    ex = {}
    for l in range(L):
        for e in range(E):
            p = (l * E + e) % n_phys
            if p not in store:
                store[p] = wl.expert_weights(gen, l, e, threads=16)
            ex[(l, e)] = store[p]
    r = make_runner(cfg, ex)
    tr = wl.routing_trace(cfg, n_steps)
    sim = CacheSim(L, E, cfg.n_slots, cfg.expert_bytes, cfg.horizon)
    nv = n_steps * L
    look = L if cfg.horizon <= 0 else cfg.horizon
    window = lambda v: tr.predicted[v + 1:min(nv, v + 1 + look)]
    w0 = window(-1)
    sim.prefetch(-1, w0); r.ctx.ef_cache_prefetch(-1, w0)
    wrs = [wl.router_weight(cfg, l) for l in range(L)]
    bufs = [torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16, device="cuda") for _ in range(2)]
    free = [int(t) for t in sample_tokens]
    forced = [int(t) for t in forced_tokens]
    assert not set(free) & set(forced)
    tok = np.asarray(free + forced)
    n_free = len(free)
    forced_dev = torch.as_tensor(forced, dtype=torch.long, device="cuda")
    worst = {"free": 0.0, "forced": 0.0}
    free_err, free_max = np.zeros(L), np.zeros(L)
    for s in range(n_steps):
        h0 = wl.activations(cfg, s)
        hd = dev_bf16(h0)
        h_ref = h0[tok]                                         # the oracle's own chain, sampled tokens only
        for l in range(L):
            v = s * L + l
            bias = wl.trace_bias(cfg, tr, v)
            win = window(v)
            dst = bufs[l & 1]
            if forced and l > 0:
                hd[forced_dev] = dev_bf16(h_ref[n_free:])        # oracle -> GPU, never the other way
            r.visit(v, hd, dst, token_bias=torch.from_numpy(bias).cuda(), predicted_next=win if len(win) else None,
                    residual=hd if L > 1 else None, pre_norm_eps=1e-5 if L > 1 else None)
            counts = np.bincount(tr.sets[v].ravel(), minlength=E)
            sim.visit(v, counts)
            if len(win):
                sim.prefetch(v, win)
            assert_cache_equal(r, sim)
            assert np.array_equal(r.counts.cpu().numpy(), counts)             # the trace bias drove the router
            # same expert SET per token as the trace intends (the order inside the set follows the natural logits)
            assert np.array_equal(np.sort(r.topk_idx[:cfg.T].cpu().numpy(), axis=1), np.sort(tr.sets[v], axis=1))
            if L > 1:
                u = oracle.round_bf16(oracle.rmsnorm(h_ref, 1e-5))
                ref = oracle.layer_forward(u, wrs[l], bias[tok], lambda e, l=l: ex[(l, e)], k, cfg.renorm, res=h_ref)
                h_ref = oracle.round_bf16(ref.out)
            else:
                ref = oracle.layer_forward(h_ref, wrs[l], bias[tok], lambda e, l=l: ex[(l, e)], k, cfg.renorm)
            r.ctx.ef_sync()
            got = bf(to_bits(dst))[tok]
            if forced:
                _, m = check_float(got[n_free:], ref.out[n_free:])
                worst["forced"] = max(worst["forced"], m)
            if free and L > 1:
                # free-running tokens: measured, not assumed -- the error after every layer goes into free_err
                fr, rf = got[:n_free], ref.out[:n_free]
                free_err[l] = max(free_err[l], np.abs(fr - rf).sum() / np.abs(rf).sum())
                free_max[l] = max(free_max[l], np.abs(fr - rf).max() / np.abs(rf).max())
            elif free:
                _, m = check_float(got[:n_free], ref.out[:n_free])
                worst["free"] = max(worst["free"], m)
            hd = dst
    r.ctx.ef_sync()
    st = r.ctx.ef_cache_get_stats()
    r.close()
    print(f"{cfg.name}: worst mean-rel error forced {worst['forced']:.2e}, free (single layer) {worst['free']:.2e}")
    if free and L > 1:
        print("free-running mean-rel error by layer:", " ".join(f"{e:.2e}" for e in free_err))
        print("free-running max-abs/max|ref| by layer:", " ".join(f"{e:.2e}" for e in free_max))
    return st, sim, free_err, free_max


def test_cfg3_mixtral_decode_full_size():
    cfg = wl.CONFIGS["mixtral_decode"]
    st, sim, _, _ = decode_case(cfg, n_steps=12, sample_tokens=range(cfg.T))
    assert st["hits"] + st["misses"] == st["lookups"] > 0
    assert st["bytes_h2d"] == cfg.expert_bytes * (st["ondemand_loads"] + st["prefetch_issued"])


def test_cfg5_stack_decode_full_shape():
    """32 layers x 8 experts at Mixtral shapes, 64 slots, 64 tokens; the 256 logical experts alias 16 physical host
    buffers so the test needs 5.6 GB of host memory, not 90 GB.  Two steps = 64 visits."""
    cfg = wl.CONFIGS["stack_decode"]
    st, sim, free_err, free_max = decode_case(cfg, n_steps=2, sample_tokens=[0, 9, 21, 30, 51, 58], phys=16,
                                              forced_tokens=[42, 63])
    assert st["prefetch_issued"] > 0 and st["prefetch_used"] > 0
    assert st["hits"] + st["misses"] == st["lookups"] == sim.stats["lookups"]
    # The FORCED tokens (oracle's bf16 input fed to every layer) hold the plain north_star tolerance at every layer: that
    # is the parity claim, asserted inside decode_case.  The FREE-running tokens compare two chains that each round the
    # hidden state to bf16 after every layer (the GPU's and the oracle's), so they drift apart; the drift is MEASURED at
    # every layer and asserted to behave like accumulated rounding noise, not like a defect:
    #  (1) it stays inside the per-layer tolerance times sqrt(depth) at EVERY depth (measured on B200, 6 tokens x 2 steps:
    #      2.5e-3 after layer 1, 1.2e-2 after 8, 2.6e-2 after 32 = 0.93 of the envelope);
    #  (2) it grows sub-linearly with depth -- the fitted exponent of err ~ depth^p is 0.65 (a systematic error,
    #      e.g. a biased rounding or a dropped term, accumulates with p >= 1);
    #  (3) a single layer applied to the drifted state adds no more than a fresh layer does: err[l+1] - err[l] never
    #      exceeds the first layer's own error by more than 50 %.
    L = cfg.n_layers
    depth = np.arange(1, L + 1)
    assert (free_err <= 5e-3 * np.sqrt(depth)).all(), free_err / np.sqrt(depth)
    assert (free_max <= 2e-2 * np.sqrt(depth)).all(), free_max / np.sqrt(depth)
    p_fit = np.polyfit(np.log(depth), np.log(free_err), 1)[0]
    print(f"free-running drift: err ~ depth^{p_fit:.2f}; err/envelope at the last layer {free_err[-1] / (5e-3 * np.sqrt(L)):.2f}")
    assert 0.3 <= p_fit <= 0.85, p_fit
    assert (np.diff(free_err) <= 1.5 * free_err[0]).all(), np.diff(free_err)


# ------------------------------------------------------------------------------------------------
# BASELINE.json states configs[2] "for 256 steps" and configs[4] "for 128 steps": the WHOLE traces, at reduced d_model /
# d_ff (the routing trace, the pool, the horizon and therefore every policy decision do not depend on them), with the slot
# table and all nine counters compared with the simulator after EVERY visit.
# ------------------------------------------------------------------------------------------------
def full_trace_accounting(name, horizon, d_model=128, d_ff=256, phys=8):
    base = wl.CONFIGS[name]
    cfg = wl.scaled(base, d_model=d_model, d_ff=d_ff, horizon=horizon)
    L, E, k, T, n_steps = cfg.n_layers, cfg.n_experts, cfg.top_k, cfg.T, cfg.n_steps
    assert (n_steps, T, cfg.n_slots) == (base.n_steps, base.T, base.n_slots)
    gen = wl.scaled(cfg, phys_experts=phys)
    store = {p: wl.expert_weights(gen, p // E, p % E) for p in range(phys)}
    ex = {(l, e): store[(l * E + e) % phys] for l in range(L) for e in range(E)}
    r = make_runner(cfg, ex)
    tr = wl.routing_trace(cfg, n_steps)
    sim = CacheSim(L, E, cfg.n_slots, cfg.expert_bytes, cfg.horizon)
    nv = n_steps * L
    look = L if cfg.horizon <= 0 else cfg.horizon
    window = lambda v: tr.predicted[v + 1:min(nv, v + 1 + look)]
    w0 = window(-1)
    sim.prefetch(-1, w0); r.ctx.ef_cache_prefetch(-1, w0)
    bufs = [torch.empty((T, cfg.d_model), dtype=torch.bfloat16, device="cuda") for _ in range(2)]
    lookups = 0
    for s in range(n_steps):
        hd = dev_bf16(wl.activations(cfg, s))
        for l in range(L):
            v = s * L + l
            win = window(v)
            dst = bufs[l & 1]
            r.visit(v, hd, dst, token_bias=torch.from_numpy(wl.trace_bias(cfg, tr, v)).cuda(),
                    predicted_next=win if len(win) else None, residual=hd if L > 1 else None,
                    pre_norm_eps=1e-5 if L > 1 else None)
            counts = np.bincount(tr.sets[v].ravel(), minlength=E)
            lookups += int((counts > 0).sum())
            sim.visit(v, counts)
            if len(win):
                sim.prefetch(v, win)
            assert_cache_equal(r, sim)                                        # slot table + 9 counters, every visit
            hd = dst
    r.ctx.ef_sync()
    assert np.array_equal(r.counts.cpu().numpy(), counts)                     # the trace bias drove the router to the end
    st = r.ctx.ef_cache_get_stats()
    assert st["lookups"] == lookups == st["hits"] + st["misses"] and st["ondemand_loads"] == st["misses"]
    assert st["bytes_h2d"] == cfg.expert_bytes * (st["ondemand_loads"] + st["prefetch_issued"])
    r.close()
    return cfg, st


def test_cfg3_whole_trace_256_steps_accounting():
    cfg, st = full_trace_accounting("mixtral_decode", horizon=None or wl.CONFIGS["mixtral_decode"].horizon)
    assert cfg.n_steps == 256 and st["lookups"] > 256 * 4
    assert 0.5 < st["hits"] / st["lookups"] < 0.95                  # 6 of 8 slots, ~7.8 active experts per step (S 8(d))


@pytest.mark.parametrize("horizon", [0, 1], ids=["fill", "one_visit_ahead"])
def test_cfg5_whole_trace_128_steps_accounting(horizon):
    """32 layers x 128 steps = 4096 visits, 64 tokens, 64 slots, both prefetch horizons (R10)."""
    cfg, st = full_trace_accounting("stack_decode", horizon=horizon)
    assert cfg.n_steps == 128 and cfg.n_layers == 32
    assert st["lookups"] >= 4096 * 7 and st["prefetch_issued"] > 0
