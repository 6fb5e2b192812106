"""Pins for the cache-policy simulator (oracle/cache_sim.py): the paper's worked examples
(tests/golden/*.json, each with its citation) and invariants that hold for any trace.  CPU only."""
import json
import os

import numpy as np
import pytest

import workloads as wl
from oracle.cache_sim import CacheSim

GOLD = os.path.join(os.path.dirname(__file__), "golden")
W = 1000


def ones(n, E):
    return [[1] * E for _ in range(n)]


def row(E, active):
    r = [0] * E
    for e in active:
        r[e] = 1
    return r


# ------------------------------------------------------------------------------------------------
# PLEC worked example
# ------------------------------------------------------------------------------------------------
def test_plec_worked_example():
    gld = json.load(open(os.path.join(GOLD, "plec_example.json")))
    L, E, S = gld["n_layers"], gld["n_experts"], gld["n_slots"]
    exp = gld["expected"]
    sim = CacheSim(L, E, S, W, horizon=0)
    n = sim.prefetch(-1, ones(L, E))                     # predicted path of the whole pass: all active
    assert n == exp["warmup_prefetches"] == sim.stats["prefetch_issued"]
    assert sorted({g // E for g in sim.snapshot()}) == exp["warmup_resident_layers"]
    counts = [1] * E
    # layer 0 computes, then PLEC refills
    plan = sim.visit(0, counts)
    assert plan.misses == []
    before = sim.snapshot()
    n = sim.prefetch(0, ones(L, E))
    assert n == exp["after_layer0_loads"]
    after = sim.snapshot()
    changed = [s for s in range(S) if before[s] != after[s]]
    assert {before[s] // E for s in changed} == {exp["after_layer0_victim_layer"]}
    assert {after[s] // E for s in changed} == {exp["after_layer0_prefetched_layer"]}
    for v in range(1, L):
        plan = sim.visit(v, counts)
        assert plan.misses == []
        sim.prefetch(v, ones(L, E))
    assert sim.stats["misses"] == exp["misses_over_one_pass"]
    assert sim.stats["ondemand_loads"] == 0
    assert sim.stats["hits"] == sim.stats["lookups"] == L * E


def test_plec_example_second_pass_also_missless():
    # steady state over several passes: every load is a prefetch, none on demand
    L, E, S = 4, 4, 8
    sim = CacheSim(L, E, S, W)
    sim.prefetch(-1, ones(L, E))
    for v in range(5 * L):
        assert sim.visit(v, [1] * E).misses == []
        sim.prefetch(v, ones(L, E))
    assert sim.stats["ondemand_loads"] == 0 and sim.stats["prefetch_wasted"] == 0
    assert sim.stats["prefetch_used"] == sim.stats["hits"] == 5 * L * E


# ------------------------------------------------------------------------------------------------
# step transition example
# ------------------------------------------------------------------------------------------------
def test_step_transition_example():
    gld = json.load(open(os.path.join(GOLD, "step_transition_example.json")))
    E, S = gld["n_experts"], gld["n_slots"]
    prev = [e - 1 for e in gld["prev_step_active"]]      # ids in the paper are one-based
    nxt = [e - 1 for e in gld["next_step_active"]]
    exp = gld["expected"]
    sim = CacheSim(1, E, S, W, horizon=1)
    sim.prefetch(-1, [row(E, prev)])
    plan = sim.visit(0, row(E, prev))
    assert plan.misses == [] and sorted(sim.snapshot()) == prev
    n = sim.prefetch(0, [row(E, nxt)])                    # issued during the previous step's computation
    assert n == exp["loads_during_prev_step"]
    res = set(sim.snapshot())
    assert res == set(nxt)
    assert [e + 1 for e in sorted(set(prev) & res)] == exp["retained"]
    assert [e + 1 for e in sorted(set(prev) - res)] == exp["evicted"]
    plan = sim.visit(1, row(E, nxt))
    assert len(plan.hits) == exp["next_step_hits"] and len(plan.misses) == exp["next_step_misses"]


# ------------------------------------------------------------------------------------------------
# correction victim order
# ------------------------------------------------------------------------------------------------
def test_correction_prefers_misprefetched():
    json.load(open(os.path.join(GOLD, "correction_example.json")))   # citation + scenario description
    L, E, S = 2, 4, 4
    sim = CacheSim(L, E, S, W)
    # layer 0 predicted {0,1}, actual {0,1}; layer 1 predicted {0,3} but actual {0,2}
    sim.prefetch(-1, [row(E, [0, 1]), row(E, [0, 3])])
    assert sorted(sim.snapshot()) == [0, 1, 4, 7]
    sim.visit(0, row(E, [0, 1]))
    sim.prefetch(0, [row(E, [0, 3])])                     # nothing to do: everything predicted is resident
    slot_of_wrong = sim.slot_of[1 * E + 3]
    plan = sim.visit(1, row(E, [0, 2]))
    # expert (1,2) was missed; the mis-prefetched (1,3) is replaced although completed experts (0,0),(0,1) exist
    assert plan.misses == [2]
    assert sim.slot_of[1 * E + 2] == slot_of_wrong
    assert (1 * E + 3) not in sim.slot_of and 0 in sim.slot_of and 1 in sim.slot_of
    assert sim.stats["prefetch_wasted"] == 1 and sim.stats["ondemand_loads"] == 1


def test_correction_falls_back_to_completed():
    L, E, S = 2, 4, 3
    sim = CacheSim(L, E, S, W)
    sim.prefetch(-1, [row(E, [0, 1]), row(E, [0])])       # all three slots: (0,0) (0,1) (1,0)
    sim.visit(0, row(E, [0, 1]))
    plan = sim.visit(1, row(E, [0, 2]))                   # (1,2) missed, no mis-prefetched expert anywhere
    assert plan.misses == [2]
    assert sim.stats["prefetch_wasted"] == 0
    # a completed layer-0 expert gave up its slot; the hit (1,0) was never disturbed
    assert (1 * E + 0) in sim.slot_of and len([g for g in sim.snapshot() if g // E == 0]) == 1


def test_phase_b_when_pool_is_all_hits():
    # S = 2, four active experts, two resident: the other two each wait for a completed slot (waves)
    sim = CacheSim(1, 4, 2, W)
    sim.prefetch(-1, [row(4, [0, 1, 2, 3])])
    assert sorted(sim.snapshot()) == [0, 1]
    plan = sim.visit(0, [1, 1, 1, 1])
    assert plan.hits == [0, 1] and plan.misses == [2, 3]
    assert [w[2] for w in plan.waves] == [False, False, True, True]
    assert sorted(sim.snapshot()) == [2, 3]
    assert sim.stats["ondemand_loads"] == 2 and sim.stats["evictions"] == 2


def test_single_slot_never_deadlocks():
    sim = CacheSim(2, 3, 1, W)
    g = wl.stream(0, "s1")
    for v in range(40):
        counts = (g.random(3) < 0.6).astype(int)
        sim.visit(v, counts)
        sim.prefetch(v, [list((g.random(3) < 0.5).astype(int))])
    st = sim.stats
    assert st["hits"] + st["misses"] == st["lookups"] and st["ondemand_loads"] == st["misses"]


# ------------------------------------------------------------------------------------------------
# invariants on seeded traces shaped like the decode configs
# ------------------------------------------------------------------------------------------------
def run_trace(cfg, H, n_steps, S=None, perfect=False):
    tr = wl.routing_trace(cfg, n_steps)
    L, E = cfg.n_layers, cfg.n_experts
    sim = CacheSim(L, E, S or cfg.n_slots, W, horizon=H)
    nv = n_steps * L
    pred = tr.actual if perfect else tr.predicted
    look = L if H <= 0 else H

    def window(v):
        return [list(pred[t]) for t in range(v + 1, min(nv, v + 1 + look))]
    sim.prefetch(-1, window(-1))
    total_act = 0
    for v in range(nv):
        counts = np.bincount(tr.sets[v].ravel(), minlength=E)
        total_act += int((counts > 0).sum())
        sim.visit(v, counts)
        # invariants after every visit
        snap = sim.snapshot()
        occ = [g for g in snap if g >= 0]
        assert len(occ) == len(set(occ)) <= sim.S                      # slot table injective
        assert all(sim.slot_of[g] == s for s, g in enumerate(snap) if g >= 0)
        sim.prefetch(v, window(v))
    st = sim.stats
    assert st["lookups"] == total_act == st["hits"] + st["misses"]
    assert st["ondemand_loads"] == st["misses"]
    assert st["bytes_h2d"] == W * (st["ondemand_loads"] + st["prefetch_issued"])
    assert st["prefetch_used"] + st["prefetch_wasted"] <= st["prefetch_issued"]
    return sim


@pytest.mark.parametrize("H", [0, 1, 3])
def test_invariants_decode_single_layer(H):
    cfg = wl.scaled(wl.CONFIGS["mixtral_decode"], d_model=64, d_ff=128)
    run_trace(cfg, H, n_steps=60)


@pytest.mark.parametrize("H", [0, 1])
def test_invariants_stack(H):
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=64, d_ff=128, T=16, n_layers=6, n_slots=12)
    run_trace(cfg, H, n_steps=12)


def test_all_resident_means_no_loads_after_warmup():
    # S >= L*E: the paper's All-In-GPU case -- after warm-up nothing moves
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=64, d_ff=128, T=8, n_layers=3, n_slots=24)
    L, E = cfg.n_layers, cfg.n_experts
    sim = CacheSim(L, E, L * E, W)
    sim.prefetch(-1, ones(L, E))
    assert sim.stats["prefetch_issued"] == L * E
    tr = wl.routing_trace(cfg, 10)
    for v in range(10 * L):
        sim.visit(v, np.bincount(tr.sets[v].ravel(), minlength=E))
        sim.prefetch(v, ones(L, E))
    assert sim.stats["misses"] == 0 and sim.stats["bytes_h2d"] == W * L * E and sim.stats["evictions"] == 0


def test_perfect_prediction_two_visits_fit_means_no_misses():
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=64, d_ff=128, T=4, n_layers=4, n_slots=16)
    sim = run_trace(cfg, H=0, n_steps=15, perfect=True)    # S = 16 >= two visits' active sets (<= 8 each)
    assert sim.stats["misses"] == 0 and sim.stats["prefetch_wasted"] == 0


def test_prediction_beats_on_demand_only():
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=64, d_ff=128, T=16, n_layers=8, n_slots=16)
    with_pred = run_trace(cfg, H=0, n_steps=10)
    tr = wl.routing_trace(cfg, 10)
    od = CacheSim(cfg.n_layers, cfg.n_experts, cfg.n_slots, W)
    for v in range(10 * cfg.n_layers):
        od.visit(v, np.bincount(tr.sets[v].ravel(), minlength=cfg.n_experts))
    assert with_pred.hit_ratio() > od.hit_ratio() + 0.2


def test_evict_removes_and_counts():
    sim = CacheSim(1, 4, 4, W)
    sim.prefetch(-1, [row(4, [0, 1, 2])])
    sim.visit(0, row(4, [0]))
    sim.evict(0, [0, 1, 3])            # 0 used, 1 never-used prefetch, 3 not resident
    assert sorted(g for g in sim.snapshot() if g >= 0) == [2]
    assert sim.stats["evictions"] == 2 and sim.stats["prefetch_wasted"] == 1


def test_stale_prefetch_is_retargeted_not_reloaded():
    # R25: a mis-prefetched expert predicted again keeps its slot and moves no bytes
    sim = CacheSim(1, 4, 2, W, horizon=1)
    sim.prefetch(-1, [row(4, [0, 1])])
    sim.visit(0, row(4, [0]))                      # expert 1 was mis-prefetched
    b = sim.stats["bytes_h2d"]
    sim.prefetch(0, [row(4, [0, 1])])              # ... and is predicted again
    assert sim.stats["bytes_h2d"] == b
    plan = sim.visit(1, row(4, [0, 1]))
    assert plan.misses == [] and sim.stats["prefetch_used"] == 2


# ------------------------------------------------------------------------------------------------
# baseline policies: LRU over the pool, LRU inside a per-layer share
# ------------------------------------------------------------------------------------------------
def one_hot_counts(E, e):
    c = [0] * E
    c[e] = 1
    return c


def test_lru_matches_the_textbook_reference_string():
    """The classic page-replacement reference string (20 references, 3 frames): LRU takes 12 faults -- one access
    per visit, so the batch semantics (hits before misses) play no part."""
    ref = [7, 0, 1, 2, 0, 3, 0, 4, 2, 3, 0, 3, 2, 1, 2, 0, 1, 7, 0, 1]
    sim = CacheSim(1, 8, 3, W, policy="lru")
    for v, e in enumerate(ref):
        sim.visit(v, one_hot_counts(8, e))
    assert sim.stats["misses"] == 12 and sim.stats["hits"] == 8
    assert sim.stats["ondemand_loads"] == 12 and sim.stats["evictions"] == 9       # 3 cold loads evict nothing
    assert sim.stats["bytes_h2d"] == 12 * W and sim.stats["prefetch_issued"] == 0
    assert sorted(sim.snapshot()) == [0, 1, 7]


@pytest.mark.parametrize("policy,L", [("lru", 1), ("lru", 3), ("layer_lru", 3)])
def test_lru_against_an_independent_ordered_dict(policy, L):
    from collections import OrderedDict
    E, S, n = 12, 6, 400
    g = np.random.default_rng(3)
    seq = g.integers(0, E, size=n)
    sim = CacheSim(L, E, S, W, policy=policy)
    sim.prefetch(-1, ones(4, E))                                   # ignored by the baselines
    caches = [OrderedDict() for _ in range(L if policy == "layer_lru" else 1)]
    cap = S // L if policy == "layer_lru" else S
    misses = 0
    for v, e in enumerate(seq):
        layer = v % L
        sim.visit(v, one_hot_counts(E, int(e)))
        c = caches[layer if policy == "layer_lru" else 0]
        key = layer * E + int(e)
        if key in c:
            c.move_to_end(key)
        else:
            misses += 1
            if len(c) >= cap:
                c.popitem(last=False)
            c[key] = True
    assert sim.stats["misses"] == misses and sim.stats["prefetch_issued"] == 0
    assert sorted(x for x in sim.snapshot() if x >= 0) == sorted(k for c in caches for k in c)
    if policy == "layer_lru":                                      # every layer stays inside its own share
        snap = sim.snapshot()
        for s, gid in enumerate(snap):
            assert gid < 0 or gid // E == s // (S // L)


def test_lru_batch_visit_never_evicts_its_own_experts_while_others_remain():
    sim = CacheSim(1, 8, 4, W, policy="lru")
    sim.visit(0, row(8, [0, 1, 2, 3]))
    plan = sim.visit(1, row(8, [2, 3, 4, 5]))                      # hits 2, 3 are locked: 4, 5 replace 0, 1
    assert plan.hits == [2, 3] and plan.misses == [4, 5]
    assert sorted(sim.snapshot()) == [2, 3, 4, 5]
    plan = sim.visit(2, row(8, [0, 1, 2, 3, 4, 5]))                # more active experts than slots: phase B reuses
    assert sim.stats["lookups"] == sim.stats["hits"] + sim.stats["misses"] == 4 + 4 + 6
    assert len(set(x for x in sim.snapshot())) == 4


def test_plec_beats_both_lru_baselines_on_the_stack_trace():
    """The paper's claim in kind (Fig. 9): with a predicted path, PLEC's hit ratio is far above on-demand LRU's."""
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=64, d_ff=128, T=16, n_layers=8, n_slots=16)
    plec = run_trace(cfg, H=1, n_steps=10)
    tr = wl.routing_trace(cfg, 10)
    for policy in ("lru", "layer_lru"):
        sim = CacheSim(cfg.n_layers, cfg.n_experts, cfg.n_slots, W, policy=policy)
        for v in range(10 * cfg.n_layers):
            sim.visit(v, np.bincount(tr.sets[v].ravel(), minlength=cfg.n_experts))
        assert plec.hit_ratio() > sim.hit_ratio() + 0.2, policy
