"""GPU parity, end to end: whole layer visits through MoELayerRunner (the public call) against the
oracle, and the cache manager's slot table + counters against oracle/cache_sim.py bit for bit."""
import numpy as np
import pytest

import oracle
import workloads as wl
from oracle.cache_sim import CacheSim, STAT_KEYS

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from test_gpu_stages import bf, check_float, dev_bf16, to_bits  # noqa: E402

EF_OPT_WAVE_BYTES, EF_OPT_CHUNK_MIN_BYTES, EF_OPT_FUSED_WAVES = 2, 3, 4      # include/ef.h


def build_runner(cfg, horizon=None, experts=None, max_tokens=None, diag=False):
    from paper_2410_17954_b200 import MoELayerRunner
    r = MoELayerRunner(cfg.n_layers, cfg.n_experts, cfg.top_k, cfg.d_model, cfg.d_ff, cfg.n_slots, cfg.n_shared,
                       max_tokens or cfg.T, cfg.horizon if horizon is None else horizon, cfg.renorm,
                       expert_kind=1 if cfg.expert_kind == "relu" else 0, diag=diag)
    experts = experts or {}
    for l in range(cfg.n_layers):
        r.set_router(l, wl.router_weight(cfg, l), wl.static_router_bias(cfg, l))
        for e in range(cfg.n_experts):
            if (l, e) not in experts:
                experts[(l, e)] = wl.expert_weights(cfg, l, e)
            r.register_expert(l, e, *experts[(l, e)])
        for s in range(cfg.n_shared):
            experts[(l, -1 - s)] = wl.expert_weights(cfg, l, -1 - s)
            r.register_expert(l, -1 - s, *experts[(l, -1 - s)])
    return r, experts


def assert_cache_equal(runner, sim):
    assert runner.ctx.ef_cache_snapshot() == sim.snapshot()
    st = runner.ctx.ef_cache_get_stats()
    assert st == {k: sim.stats[k] for k in STAT_KEYS}


# ------------------------------------------------------------------------------------------------
# cfg 1 (tiny): the whole visit, predicted path 100% correct, cold cache of 4 slots
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("simt", [True, False], ids=["simt_debug", "tcgen05"])
def test_cfg1_tiny_end_to_end(simt):
    cfg = wl.CONFIGS["tiny"]
    r, ex = build_runner(cfg, diag=simt)
    if simt:
        r.ctx.ef_diag_set_simt_ffn(True)
    x = wl.activations(cfg)
    ref = oracle.layer_forward(x, wl.router_weight(cfg), None, [ex[(0, e)] for e in range(cfg.n_experts)], cfg.top_k)
    predicted = (ref.counts > 0).astype(np.uint8)[None, :]          # "a routing path that is 100% correct"
    sim = CacheSim(1, cfg.n_experts, cfg.n_slots, cfg.expert_bytes, cfg.horizon)
    sim.prefetch(-1, predicted); r.ctx.ef_cache_prefetch(-1, predicted)
    assert_cache_equal(r, sim)
    out = torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16, device="cuda")
    r.visit(0, dev_bf16(x), out, want_logits=True)
    sim.visit(0, ref.counts)
    r.ctx.ef_sync()
    assert_cache_equal(r, sim)
    assert sim.stats["lookups"] == int((ref.counts > 0).sum())
    # integers bit-exact
    assert np.array_equal(r.topk_idx.cpu().numpy(), ref.idx)
    assert np.array_equal(r.counts.cpu().numpy(), ref.counts)
    assert np.array_equal(r.offsets.cpu().numpy(), ref.offsets)
    assert np.array_equal(r.src.cpu().numpy(), ref.src)
    assert np.array_equal(r.inv.cpu().numpy(), ref.inv)
    assert np.array_equal(to_bits(r.x_perm), ref.x_perm)
    np.testing.assert_allclose(r.topk_w.cpu().numpy(), ref.w, rtol=2e-4)
    check_float(bf(to_bits(r.y_perm)), ref.y_perm)
    check_float(bf(to_bits(out)), ref.out)
    r.close()


def test_identical_experts_reduce_to_dense_ffn_on_gpu():
    cfg = wl.scaled(wl.CONFIGS["tiny"], T=48, n_slots=8)
    w3 = wl.expert_weights(cfg, 0, 0)
    r, _ = build_runner(cfg, experts={(0, e): w3 for e in range(cfg.n_experts)})
    x = wl.activations(cfg)
    out = torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16, device="cuda")
    r.visit(0, dev_bf16(x), out)
    r.ctx.ef_sync()
    dense = oracle.expert_ffn(x, *w3)
    check_float(bf(to_bits(out)), dense)
    r.close()


# ------------------------------------------------------------------------------------------------
# shared experts + skewed many-expert routing (cfg 4 shape, reduced size)
# ------------------------------------------------------------------------------------------------
def test_cfg4_reduced_shared_experts_and_zipf():
    cfg = wl.scaled(wl.CONFIGS["many_expert_prefill"], T=512, d_model=256, d_ff=384)
    r, ex = build_runner(cfg)
    x = wl.activations(cfg)
    ref = oracle.layer_forward(x, wl.router_weight(cfg), wl.static_router_bias(cfg),
                               [ex[(0, e)] for e in range(cfg.n_experts)], cfg.top_k,
                               shared=[ex[(0, -1)], ex[(0, -2)]])
    srt = np.sort(ref.logits, axis=1)[:, ::-1]
    assert (srt[:, cfg.top_k - 1] - srt[:, cfg.top_k]).min() > 1e-5     # routing unambiguous at fp32 (R22)
    predicted = (ref.counts > 0).astype(np.uint8)[None, :]
    sim = CacheSim(1, cfg.n_experts, cfg.n_slots, cfg.expert_bytes, cfg.horizon)
    sim.prefetch(-1, predicted); r.ctx.ef_cache_prefetch(-1, predicted)
    out = torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16, device="cuda")
    r.visit(0, dev_bf16(x), out)
    sim.visit(0, ref.counts)
    r.ctx.ef_sync()
    assert np.array_equal(r.topk_idx.cpu().numpy(), ref.idx)
    assert np.array_equal(r.inv.cpu().numpy(), ref.inv)
    assert_cache_equal(r, sim)
    assert sim.stats["misses"] > 0                                       # waves were exercised
    check_float(bf(to_bits(out)), ref.out)
    r.close()


# ------------------------------------------------------------------------------------------------
# physical scheduling of on-demand loads: batched miss waves and two-chunk expert copies change
# neither the result nor the accounting -- down to pools so small that a miss takes the slot of a miss of the same visit
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_slots", [1, 2, 5, 24])
@pytest.mark.parametrize("wave_bytes,chunk_min,fused,copy_order",
                         [(0, 0, 1, 1), (1 << 40, 0, 1, 1), (0, 1, 1, 1), (1 << 40, 1, 1, 1), (None, None, 1, 1),
                          (0, 1, 0, 1), (1 << 40, 0, 0, 1), (None, None, 1, 0), (4 * 3 * 256 * 384 * 2, 0, 1, 0)],
                         ids=["single_waves", "batched", "chunked", "batched_chunked", "defaults", "chunked_two_launches",
                              "batched_two_launches", "policy_copy_order", "waves_of_4_policy_copy_order"])
def test_miss_wave_batching_and_chunked_copies(n_slots, wave_bytes, chunk_min, fused, copy_order):
    """Results, slot table and counters are identical however the on-demand loads are scheduled physically: one wave per
    miss or geometric batches, whole or two-chunk copies, one or two launches per wave, copies in policy order or with the
    most routed rows first (later 'generations' -- misses that reuse the slot of an earlier miss of the visit -- behind)."""
    cfg = wl.scaled(wl.CONFIGS["many_expert_prefill"], T=256, d_model=256, d_ff=384, n_slots=n_slots)
    r, ex = build_runner(cfg)
    r.ctx.ef_set_option(EF_OPT_FUSED_WAVES, fused)
    r.ctx.ef_set_option(6, copy_order)                   # EF_OPT_COPY_ORDER
    if wave_bytes is not None:
        r.ctx.ef_set_option(EF_OPT_WAVE_BYTES, wave_bytes)
        r.ctx.ef_set_option(EF_OPT_CHUNK_MIN_BYTES, chunk_min)
    x = wl.activations(cfg)
    ref = oracle.layer_forward(x, wl.router_weight(cfg), wl.static_router_bias(cfg),
                               [ex[(0, e)] for e in range(cfg.n_experts)], cfg.top_k,
                               shared=[ex[(0, -1)], ex[(0, -2)]])
    predicted = (ref.counts > 0).astype(np.uint8)[None, :]
    sim = CacheSim(1, cfg.n_experts, cfg.n_slots, cfg.expert_bytes, cfg.horizon)
    sim.prefetch(-1, predicted); r.ctx.ef_cache_prefetch(-1, predicted)
    out = torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16, device="cuda")
    for v in range(2):                                   # the second visit starts from a full pool
        r.visit(v, dev_bf16(x), out)
        sim.visit(v, ref.counts)
        r.ctx.ef_sync()
        assert_cache_equal(r, sim)
        assert np.array_equal(r.inv.cpu().numpy(), ref.inv)
        check_float(bf(to_bits(out)), ref.out)
    assert sim.stats["misses"] > n_slots
    r.close()


# ------------------------------------------------------------------------------------------------
# Switch-style layer (f4, R30): top-1, full-softmax gate weight (Eq. 2), ReLU experts, Zipf skew, 16 of 64 slots
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T", [512, 4096], ids=["reduced", "full_size_switch_prefill"])
def test_switch_prefill_relu_top1(T):
    cfg = wl.scaled(wl.CONFIGS["switch_prefill"], T=T)
    r, ex = build_runner(cfg)
    x = wl.activations(cfg)
    wr, bias = wl.router_weight(cfg), wl.static_router_bias(cfg)
    g = np.random.default_rng(T)
    rows = None if T <= 512 else np.sort(g.choice(T, 96, replace=False))
    ref = oracle.layer_forward(x, wr, bias, [ex[(0, e)] for e in range(cfg.n_experts)], 1, renorm=0, rows=rows)
    predicted = (ref.counts > 0).astype(np.uint8)[None, :]
    sim = CacheSim(1, cfg.n_experts, cfg.n_slots, cfg.expert_bytes)
    assert cfg.expert_bytes == 2 * cfg.d_model * cfg.d_ff * 2
    sim.prefetch(-1, predicted); r.ctx.ef_cache_prefetch(-1, predicted)
    out = torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16, device="cuda")
    r.visit(0, dev_bf16(x), out, want_logits=True)
    sim.visit(0, ref.counts)
    r.ctx.ef_sync()
    # top-1 decided on identical logits (R22): the oracle's argmax applied to the GPU's own logits
    gl = r.logits.cpu().numpy()[:T].astype(np.float64)
    idx_ref, w_ref = oracle.topk_gate(gl, 1, renorm=0)
    assert np.array_equal(r.topk_idx.cpu().numpy()[:T], idx_ref)
    assert np.array_equal(r.topk_idx.cpu().numpy()[:T], ref.idx)          # and the generator's logit gap holds
    assert np.allclose(r.topk_w.cpu().numpy()[:T], w_ref, rtol=1e-5)
    assert np.array_equal(r.inv.cpu().numpy()[:T], ref.inv)
    assert_cache_equal(r, sim)
    assert sim.stats["bytes_h2d"] == cfg.expert_bytes * (sim.stats["ondemand_loads"] + sim.stats["prefetch_issued"])
    if T == wl.CONFIGS["switch_prefill"].T:
        assert sim.stats["misses"] > 0                                    # more active experts than slots: waves ran
    got = bf(to_bits(out))
    check_float(got if rows is None else got[rows], ref.out)
    r.close()


# ------------------------------------------------------------------------------------------------
# decode traces: cache accounting bit-exact over many visits; outputs checked on sampled visits
# ------------------------------------------------------------------------------------------------
def run_decode(cfg, n_steps, horizon, check_out_every, policy="plec", early_release=None, launches=None, splitk=None):
    L, E = cfg.n_layers, cfg.n_experts
    r, ex = build_runner(cfg, horizon=horizon)
    r.ctx.ef_set_cache_policy(policy)
    if early_release is not None:
        r.ctx.ef_set_option(7, early_release)             # EF_OPT_EARLY_RELEASE
    if splitk is not None:
        r.ctx.ef_set_option(1, splitk)                    # EF_OPT_SPLITK
    tr = wl.routing_trace(cfg, n_steps)
    sim = CacheSim(L, E, cfg.n_slots, cfg.expert_bytes, horizon, policy=policy)
    nv = n_steps * L
    look = L if horizon <= 0 else horizon

    def window(v):
        return tr.predicted[v + 1:min(nv, v + 1 + look)]
    w0 = window(-1)
    sim.prefetch(-1, w0); r.ctx.ef_cache_prefetch(-1, w0)
    out = torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16, device="cuda")
    wrs = [wl.router_weight(cfg, l) for l in range(L)]
    for s in range(n_steps):
        h = wl.activations(cfg, s)                       # fresh seeded h_0 per step
        hd = dev_bf16(h)
        for l in range(L):
            v = s * L + l
            bias = wl.trace_bias(cfg, tr, v)
            win = window(v)
            nxt = torch.empty_like(hd)
            r.visit(v, hd, nxt, token_bias=torch.from_numpy(bias).cuda(), predicted_next=win if len(win) else None,
                    residual=hd if L > 1 else None, pre_norm_eps=1e-5 if L > 1 else None)
            counts = np.bincount(tr.sets[v].ravel(), minlength=E)
            sim.visit(v, counts)
            if len(win):
                sim.prefetch(v, win)
            assert_cache_equal(r, sim)
            check = check_out_every and v % check_out_every == 0
            if L > 1:
                # the oracle runs its own chain from the seeded h_0 (nothing flows from the GPU into it);
                # activations between layers are bf16 at the boundary, so it rounds exactly there
                u = oracle.round_bf16(oracle.rmsnorm(h, 1e-5))
                ref = oracle.layer_forward(u, wrs[l], bias, [ex[(l, e)] for e in range(E)], cfg.top_k, res=h)
                h = oracle.round_bf16(ref.out)
            elif check:
                ref = oracle.layer_forward(h, wrs[l], bias, [ex[(l, e)] for e in range(E)], cfg.top_k)
            if check:
                r.ctx.ef_sync()
                assert np.array_equal(r.counts.cpu().numpy(), counts)          # the trace bias drove the router
                assert np.array_equal(r.topk_idx.cpu().numpy(), ref.idx)
                check_float(bf(to_bits(nxt)), ref.out)
            hd = nxt
    r.ctx.ef_sync()
    st = r.ctx.ef_cache_get_stats()
    if launches is not None:
        launches.append(r.ctx.ef_launch_count())
    r.close()
    return st, sim


@pytest.mark.parametrize("d_model,d_ff,T,splitk", [(256, 512, 16, None), (512, 3072, 16, None), (256, 512, 100, 1)],
                         ids=["short_k", "long_k_split", "wider_tiles_no_split"])
def test_first_victim_slot_is_handed_back_from_inside_the_hits_wave(d_model, d_ff, T, splitk):
    """EF_OPT_EARLY_RELEASE: the hit whose slot the first pending copy overwrites runs inside the hits' wave (ticketed first)
    and the copy waits on a device word its GEMM2 units bump, instead of on the event behind a launch of its own.  The
    copy then lands in the slot WHILE that wave is still running: outputs are checked against the oracle after every
    visit (a hand-back that came too early would feed the rest of the wave the next expert's weights), the slot table and
    the counters are the simulator's with the option on and off, and with it on there are fewer launches.  (A wave hands a
    slot back only when the first victim is a decode-sized expert: one token tile of <= 128 rows.)"""
    cfg = wl.scaled(wl.CONFIGS["mixtral_decode"], d_model=d_model, d_ff=d_ff, T=T)
    n = {}
    for on in (1, 0):
        L = []
        st, sim = run_decode(cfg, n_steps=24, horizon=1, check_out_every=1, early_release=on, launches=L, splitk=splitk)
        n[on] = (L[0], st)
    assert n[1][1] == n[0][1]                   # accounting does not depend on the physical schedule
    assert n[1][0] < n[0][0], n                 # the early path really ran: one launch fewer per visit with a first victim


@pytest.mark.parametrize("horizon", [1, 0])
def test_cfg3_reduced_decode_trace(horizon):
    cfg = wl.scaled(wl.CONFIGS["mixtral_decode"], d_model=256, d_ff=512)
    st, sim = run_decode(cfg, n_steps=48, horizon=horizon, check_out_every=7)
    assert st["lookups"] > 0 and st["hits"] + st["misses"] == st["lookups"]
    assert st["bytes_h2d"] == cfg.expert_bytes * (st["ondemand_loads"] + st["prefetch_issued"])


@pytest.mark.parametrize("horizon", [0, 1])
def test_cfg5_reduced_stack_trace(horizon):
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=256, d_ff=512, T=32, n_layers=6, n_slots=12)
    st, sim = run_decode(cfg, n_steps=10, horizon=horizon, check_out_every=5)
    assert st["prefetch_issued"] > 0 and st["misses"] < st["lookups"]


def test_long_trace_wraps_the_event_ring():
    """More loads and waves than the library's ring of 2048 sync events holds (handles are recycled, a stale handle
    degrades to 'wait for everything enqueued so far'): accounting bit-exact at every visit and outputs on sampled
    visits stay right over ~1000 visits with chunked copies forced on."""
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=256, d_ff=512, T=32, n_layers=6, n_slots=12)
    L, E = cfg.n_layers, cfg.n_experts
    n_steps = 170
    r, ex = build_runner(cfg, horizon=0)
    r.ctx.ef_set_option(EF_OPT_CHUNK_MIN_BYTES, 1)                      # two copies + two ready events per load
    r.ctx.ef_set_option(EF_OPT_WAVE_BYTES, 0)                           # one wave (and one free event) per miss
    tr = wl.routing_trace(cfg, n_steps)
    sim = CacheSim(L, E, cfg.n_slots, cfg.expert_bytes, 0)
    nv = n_steps * L
    window = lambda v: tr.predicted[v + 1:min(nv, v + 1 + L)]
    sim.prefetch(-1, window(-1)); r.ctx.ef_cache_prefetch(-1, window(-1))
    wrs = [wl.router_weight(cfg, l) for l in range(L)]
    for s in range(n_steps):
        h = wl.activations(cfg, s)
        hd = dev_bf16(h)
        check = s % 40 == 39
        for l in range(L):
            v = s * L + l
            bias = wl.trace_bias(cfg, tr, v)
            win = window(v)
            nxt = torch.empty_like(hd)
            r.visit(v, hd, nxt, token_bias=torch.from_numpy(bias).cuda(), predicted_next=win if len(win) else None,
                    residual=hd, pre_norm_eps=1e-5)
            sim.visit(v, np.bincount(tr.sets[v].ravel(), minlength=E))
            if len(win):
                sim.prefetch(v, win)
            if check:
                u = oracle.round_bf16(oracle.rmsnorm(h, 1e-5))
                ref = oracle.layer_forward(u, wrs[l], bias, [ex[(l, e)] for e in range(E)], cfg.top_k, res=h)
                h = oracle.round_bf16(ref.out)
            hd = nxt
        assert_cache_equal(r, sim)
        if check:
            r.ctx.ef_sync()
            check_float(bf(to_bits(hd)), bf(h))
    st = r.ctx.ef_cache_get_stats()
    assert 2 * (st["ondemand_loads"] + st["prefetch_issued"]) > 2 * 2048      # the ring went round at least twice
    r.close()


@pytest.mark.parametrize("policy", ["lru", "layer_lru"])
def test_baseline_policies_match_simulator(policy):
    """the LRU baselines in the library against the simulator, slot table and counters bit-exact at
    every visit, outputs on sampled visits; predictions are supplied and ignored."""
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=256, d_ff=512, T=32, n_layers=6, n_slots=12)
    st, sim = run_decode(cfg, n_steps=8, horizon=1, check_out_every=5, policy=policy)
    assert st["prefetch_issued"] == 0 and st["misses"] == st["ondemand_loads"] > 0
    assert st["bytes_h2d"] == cfg.expert_bytes * st["ondemand_loads"]


def test_cache_policy_can_only_change_on_an_empty_table():
    from paper_2410_17954_b200 import EfError
    cfg = wl.scaled(wl.CONFIGS["tiny"], n_slots=6)
    r, _ = build_runner(cfg)
    r.ctx.ef_cache_prefetch(-1, np.ones((1, cfg.n_experts), np.uint8))
    with pytest.raises(EfError):
        r.ctx.ef_set_cache_policy("lru")
    r.ctx.ef_cache_clear()
    r.ctx.ef_set_cache_policy("lru")
    with pytest.raises(EfError):
        r.ctx.ef_set_cache_policy(7)
    r.close()


def test_evict_and_clear_match_simulator():
    cfg = wl.scaled(wl.CONFIGS["tiny"], n_slots=6)
    r, _ = build_runner(cfg)
    sim = CacheSim(1, cfg.n_experts, cfg.n_slots, cfg.expert_bytes)
    p = np.array([[1, 1, 0, 1, 1, 0, 1, 0]], np.uint8)
    sim.prefetch(-1, p); r.ctx.ef_cache_prefetch(-1, p)
    sim.evict(0, [1, 2, 4]); r.ctx.ef_cache_evict(0, [1, 2, 4])
    assert_cache_equal(r, sim)
    r.ctx.ef_cache_clear()
    assert r.ctx.ef_cache_snapshot() == [-1] * cfg.n_slots
    r.close()


# ------------------------------------------------------------------------------------------------
# boundary behaviour stated in include/ef.h
# ------------------------------------------------------------------------------------------------
def test_permute_with_caller_mirror_then_ffn_with_null_counts():
    """ef.h (ef_permute): with a caller-supplied pinned mirror the internal event is still recorded, and
    ef_expert_ffn_grouped(counts_host = NULL) waits on it and reads THAT mirror."""
    cfg = wl.scaled(wl.CONFIGS["tiny"], n_slots=8)
    r, ex = build_runner(cfg)
    x = wl.activations(cfg)
    ref = oracle.layer_forward(x, wl.router_weight(cfg), None, [ex[(0, e)] for e in range(cfg.n_experts)], cfg.top_k)
    c, T = r.ctx, cfg.T
    xd = dev_bf16(x)
    mine = torch.full((cfg.n_experts,), -7, dtype=torch.int32).pin_memory()
    out = torch.empty((T, cfg.d_model), dtype=torch.bfloat16, device="cuda")
    for rep in range(2):                                  # the second pass must not see the first pass's event / mirror
        mine.fill_(-7)
        c.ef_route_topk(xd, r.w_router[0], None, T, 1, r.topk_idx, r.topk_w, None)
        c.ef_permute(r.topk_idx, xd, T, r.x_perm, r.counts, r.offsets, r.src, r.inv, mine)
        c.ef_expert_ffn_grouped(rep, 0, r.x_perm, None, r.y_perm)
        assert np.array_equal(mine.numpy(), ref.counts)   # the call waited for the mirror
        c.ef_combine(r.y_perm, r.inv, r.topk_w, T, None, None, out)
        c.ef_sync()
        check_float(bf(to_bits(out)), ref.out)
    assert c.ef_cache_get_stats()["lookups"] == 2 * int((ref.counts > 0).sum())
    r.close()


def test_out_of_range_topk_index_is_skipped_and_flagged():
    """ef.h (ef_permute): a top-k index outside [0, E) is routed nowhere (inv = -1, left out of every count) and the
    next ef_expert_ffn_grouped(counts_host = NULL) refuses to run; ef_combine skips the pair."""
    from paper_2410_17954_b200 import EfError
    cfg = wl.scaled(wl.CONFIGS["tiny"], n_slots=8)
    r, ex = build_runner(cfg)
    T, k, E = cfg.T, cfg.top_k, cfg.n_experts
    g = np.random.default_rng(0)
    idx = np.stack([g.choice(E, k, replace=False) for _ in range(T)]).astype(np.int32)
    bad = [(3, 0, E), (40, 1, -1), (63, 1, 1 << 20)]
    for t, j, v in bad:
        idx[t, j] = v
    xd = dev_bf16(wl.activations(cfg))
    r.topk_idx.copy_(torch.from_numpy(idx))
    r.ctx.ef_permute(r.topk_idx, xd, T, r.x_perm, r.counts, r.offsets, r.src, r.inv)
    torch.cuda.synchronize()
    good = np.ones((T, k), bool)
    for t, j, _ in bad:
        good[t, j] = False
    counts_ref = np.bincount(idx[good], minlength=E)
    assert np.array_equal(r.counts.cpu().numpy(), counts_ref)
    inv = r.inv.cpu().numpy().reshape(T, k)
    assert (inv[~good] == -1).all() and sorted(inv[good]) == list(range(int(counts_ref.sum())))
    with pytest.raises(EfError) as e:
        r.ctx.ef_expert_ffn_grouped(0, 0, r.x_perm, None, r.y_perm)
    assert e.value.code == -1
    r.y_perm.zero_(); r.topk_w.fill_(1.0)
    out = torch.empty((T, cfg.d_model), dtype=torch.bfloat16, device="cuda")
    r.ctx.ef_combine(r.y_perm, r.inv, r.topk_w, T, None, None, out)       # must not read row -1
    r.ctx.ef_sync()
    assert float(out.float().abs().max()) == 0.0
    r.close()


def test_nan_activations_still_route_to_valid_experts():
    """R2: NaN logits are undefined input, but the router must never emit an index outside [0, E): a NaN logit ranks as
    -inf and the lowest untaken index wins, exactly what the oracle's strict '>' scan does on an all-NaN row."""
    cfg = wl.scaled(wl.CONFIGS["tiny"], n_slots=8)
    r, _ = build_runner(cfg)
    T, k, E = cfg.T, cfg.top_k, cfg.n_experts
    x = bf(wl.activations(cfg)).astype(np.float32)
    x[5, :] = np.nan
    xd = torch.from_numpy(x).cuda().to(torch.bfloat16)
    r.ctx.ef_route_topk(xd, r.w_router[0], None, T, 1, r.topk_idx, r.topk_w, r.logits)
    torch.cuda.synchronize()
    idx = r.topk_idx.cpu().numpy()
    assert idx.min() >= 0 and idx.max() < E
    assert list(idx[5]) == list(range(k))
    idx_ref, _ = oracle.topk_gate(r.logits.cpu().numpy().astype(np.float64), k, 1)
    assert np.array_equal(idx, idx_ref)
    r.ctx.ef_permute(r.topk_idx, xd, T, r.x_perm, r.counts, r.offsets, r.src, r.inv)
    r.ctx.ef_sync()
    assert int(r.counts.sum()) == T * k
    r.close()


def test_calls_on_a_second_stream_are_ordered_behind_the_first():
    """ef.h (Streams): the layer calls share per-ctx workspaces; a call on another stream is serialised behind what the
    lane has enqueued so far.  Two visits on two streams, no host synchronisation in between."""
    cfg = wl.scaled(wl.CONFIGS["tiny"], T=64, d_model=512, d_ff=1024, n_slots=8)
    r, ex = build_runner(cfg)
    x = wl.activations(cfg)
    ref = oracle.layer_forward(x, wl.router_weight(cfg), None, [ex[(0, e)] for e in range(cfg.n_experts)], cfg.top_k)
    xd = dev_bf16(x)
    outs = [torch.empty((cfg.T, cfg.d_model), dtype=torch.bfloat16, device="cuda") for _ in range(6)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    for v in range(6):
        with torch.cuda.stream(streams[v & 1]):
            r.visit(v, xd, outs[v])
    r.ctx.ef_sync()
    for o in outs:
        check_float(bf(to_bits(o)), ref.out)
    r.close()


def test_reregistering_a_resident_or_aliased_expert_is_refused():
    from paper_2410_17954_b200 import EfError
    cfg = wl.scaled(wl.CONFIGS["tiny"], n_slots=4)
    r, ex = build_runner(cfg)
    c = r.ctx
    c.ef_host_expert_alias(0, 7, 0, 2)                       # expert 7 now shares expert 2's packed host buffer
    with pytest.raises(EfError):
        c.ef_host_expert_register(0, 2, *ex[(0, 2)])         # would pull the buffer from under the alias
    c.ef_cache_prefetch(-1, np.array([[1, 0, 0, 0, 0, 0, 0, 0]], np.uint8))
    with pytest.raises(EfError):
        c.ef_host_expert_register(0, 0, *ex[(0, 0)])         # resident: the slot would keep serving the old weights
    c.ef_cache_evict(0, [0])
    c.ef_host_expert_register(0, 0, *ex[(0, 1)])             # evicted: allowed (waits for the copy stream first)
    c.ef_host_expert_register(0, 7, *ex[(0, 7)])             # an alias may become an owner again ...
    c.ef_host_expert_register(0, 2, *ex[(0, 2)])             # ... which frees its former source for re-registration
    r.close()


def test_memory_bound_calls_can_be_captured_into_a_cuda_graph():
    """ef.h (CUDA graphs): rmsnorm -> route -> permute and combine, captured once and replayed, give what the eager calls
    give; a captured ef_permute leaves no counts mirror behind."""
    from paper_2410_17954_b200 import EfError
    cfg = wl.scaled(wl.CONFIGS["tiny"], n_slots=8)
    r, ex = build_runner(cfg)
    c, T = r.ctx, cfg.T
    x = dev_bf16(wl.activations(cfg))
    normed = torch.empty_like(x)
    out_e = torch.empty_like(x); out_g = torch.empty_like(x)

    def front():
        c.ef_rmsnorm(x, T, 1e-5, normed)
        c.ef_route_topk(normed, r.w_router[0], None, T, 1, r.topk_idx, r.topk_w, None)
        c.ef_permute(r.topk_idx, normed, T, r.x_perm, r.counts, r.offsets, r.src, r.inv)
    front()
    c.ef_expert_ffn_grouped(0, 0, r.x_perm, None, r.y_perm)
    c.ef_combine(r.y_perm, r.inv, r.topk_w, T, x, None, out_e)
    c.ef_sync()
    eager = [t.clone() for t in (r.topk_idx, r.topk_w, r.counts, r.offsets, r.src, r.inv, r.x_perm)]
    for t in (r.topk_idx, r.counts, r.offsets, r.src, r.inv):
        t.fill_(-1)
    r.x_perm.zero_()
    g1, g2 = torch.cuda.CUDAGraph(), torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    with torch.cuda.graph(g1, stream=s):
        front()
    with pytest.raises(EfError):                       # nothing ran: there is no mirror to wait for
        c.ef_expert_ffn_grouped(1, 0, r.x_perm, None, r.y_perm)
    with torch.cuda.graph(g2, stream=s):
        c.ef_combine(r.y_perm, r.inv, r.topk_w, T, x, None, out_g)
    g1.replay()
    torch.cuda.synchronize()
    for a, b in zip(eager, (r.topk_idx, r.topk_w, r.counts, r.offsets, r.src, r.inv, r.x_perm)):
        assert torch.equal(a, b)
    g2.replay()
    torch.cuda.synchronize()
    assert torch.equal(out_e, out_g)
    r.close()
