"""Pins for the cache-policy simulator (oracle/cache_sim.py): the paper's worked examples
(tests/golden/*.json, each with its citation) and invariants that hold for any trace.  CPU only."""
import json
import os

import numpy as np
import pytest

import workloads as wl
from oracle.cache_sim import CacheSim, belady_min_loads

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
def test_plec_worked_example(Sim=CacheSim):
    gld = json.load(open(os.path.join(GOLD, "plec_example.json")))
    L, E, S = gld["n_layers"], gld["n_experts"], gld["n_slots"]
    exp = gld["expected"]
    sim = Sim(L, E, S, W, horizon=0)
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


def test_plec_example_second_pass_also_missless(Sim=CacheSim):
    # steady state over several passes: every load is a prefetch, none on demand
    L, E, S = 4, 4, 8
    sim = Sim(L, E, S, W)
    sim.prefetch(-1, ones(L, E))
    for v in range(5 * L):
        assert sim.visit(v, [1] * E).misses == []
        sim.prefetch(v, ones(L, E))
    assert sim.stats["ondemand_loads"] == 0 and sim.stats["prefetch_wasted"] == 0
    assert sim.stats["prefetch_used"] == sim.stats["hits"] == 5 * L * E


# ------------------------------------------------------------------------------------------------
# step transition example
# ------------------------------------------------------------------------------------------------
def test_step_transition_example(Sim=CacheSim):
    gld = json.load(open(os.path.join(GOLD, "step_transition_example.json")))
    E, S = gld["n_experts"], gld["n_slots"]
    prev = [e - 1 for e in gld["prev_step_active"]]      # ids in the paper are one-based
    nxt = [e - 1 for e in gld["next_step_active"]]
    exp = gld["expected"]
    sim = Sim(1, E, S, W, horizon=1)
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
def test_correction_prefers_misprefetched(Sim=CacheSim):
    json.load(open(os.path.join(GOLD, "correction_example.json")))   # citation + scenario description
    L, E, S = 2, 4, 4
    sim = Sim(L, E, S, W)
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


def test_correction_falls_back_to_completed(Sim=CacheSim):
    L, E, S = 2, 4, 3
    sim = Sim(L, E, S, W)
    sim.prefetch(-1, [row(E, [0, 1]), row(E, [0])])       # all three slots: (0,0) (0,1) (1,0)
    sim.visit(0, row(E, [0, 1]))
    plan = sim.visit(1, row(E, [0, 2]))                   # (1,2) missed, no mis-prefetched expert anywhere
    assert plan.misses == [2]
    assert sim.stats["prefetch_wasted"] == 0
    # a completed layer-0 expert gave up its slot; the hit (1,0) was never disturbed
    assert (1 * E + 0) in sim.slot_of and len([g for g in sim.snapshot() if g // E == 0]) == 1


def test_phase_b_when_pool_is_all_hits(Sim=CacheSim):
    # S = 2, four active experts, two resident: the other two each wait for a completed slot (waves)
    sim = Sim(1, 4, 2, W)
    sim.prefetch(-1, [row(4, [0, 1, 2, 3])])
    assert sorted(sim.snapshot()) == [0, 1]
    plan = sim.visit(0, [1, 1, 1, 1])
    assert plan.hits == [0, 1] and plan.misses == [2, 3]
    assert [w[2] for w in plan.waves] == [False, False, True, True]
    assert sorted(sim.snapshot()) == [2, 3]
    assert sim.stats["ondemand_loads"] == 2 and sim.stats["evictions"] == 2


def test_single_slot_never_deadlocks(Sim=CacheSim):
    sim = Sim(2, 3, 1, W)
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
def run_trace(cfg, H, n_steps, S=None, perfect=False, Sim=CacheSim):
    tr = wl.routing_trace(cfg, n_steps)
    L, E = cfg.n_layers, cfg.n_experts
    sim = Sim(L, E, S or cfg.n_slots, W, horizon=H)
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
def test_invariants_decode_single_layer(H, Sim=CacheSim):
    cfg = wl.scaled(wl.CONFIGS["mixtral_decode"], d_model=64, d_ff=128)
    run_trace(cfg, H, n_steps=60, Sim=Sim)


@pytest.mark.parametrize("H", [0, 1])
def test_invariants_stack(H, Sim=CacheSim):
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=64, d_ff=128, T=16, n_layers=6, n_slots=12)
    run_trace(cfg, H, n_steps=12, Sim=Sim)


def test_all_resident_means_no_loads_after_warmup(Sim=CacheSim):
    # S >= L*E: the paper's All-In-GPU case -- after warm-up nothing moves
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=64, d_ff=128, T=8, n_layers=3, n_slots=24)
    L, E = cfg.n_layers, cfg.n_experts
    sim = Sim(L, E, L * E, W)
    sim.prefetch(-1, ones(L, E))
    assert sim.stats["prefetch_issued"] == L * E
    tr = wl.routing_trace(cfg, 10)
    for v in range(10 * L):
        sim.visit(v, np.bincount(tr.sets[v].ravel(), minlength=E))
        sim.prefetch(v, ones(L, E))
    assert sim.stats["misses"] == 0 and sim.stats["bytes_h2d"] == W * L * E and sim.stats["evictions"] == 0


def test_perfect_prediction_two_visits_fit_means_no_misses(Sim=CacheSim):
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=64, d_ff=128, T=4, n_layers=4, n_slots=16)
    sim = run_trace(cfg, H=0, n_steps=15, perfect=True, Sim=Sim)    # S = 16 >= two visits' active sets (<= 8 each)
    assert sim.stats["misses"] == 0 and sim.stats["prefetch_wasted"] == 0


def test_prediction_beats_on_demand_only(Sim=CacheSim):
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=64, d_ff=128, T=16, n_layers=8, n_slots=16)
    with_pred = run_trace(cfg, H=0, n_steps=10, Sim=Sim)
    tr = wl.routing_trace(cfg, 10)
    od = Sim(cfg.n_layers, cfg.n_experts, cfg.n_slots, W)
    for v in range(10 * cfg.n_layers):
        od.visit(v, np.bincount(tr.sets[v].ravel(), minlength=cfg.n_experts))
    assert with_pred.hit_ratio() > od.hit_ratio() + 0.2


def test_evict_removes_and_counts(Sim=CacheSim):
    sim = Sim(1, 4, 4, W)
    sim.prefetch(-1, [row(4, [0, 1, 2])])
    sim.visit(0, row(4, [0]))
    sim.evict(0, [0, 1, 3])            # 0 used, 1 never-used prefetch, 3 not resident
    assert sorted(g for g in sim.snapshot() if g >= 0) == [2]
    assert sim.stats["evictions"] == 2 and sim.stats["prefetch_wasted"] == 1


def test_stale_prefetch_is_retargeted_not_reloaded(Sim=CacheSim):
    # R25: a mis-prefetched expert predicted again keeps its slot and moves no bytes
    sim = Sim(1, 4, 2, W, horizon=1)
    sim.prefetch(-1, [row(4, [0, 1])])
    sim.visit(0, row(4, [0]))                      # expert 1 was mis-prefetched
    b = sim.stats["bytes_h2d"]
    sim.prefetch(0, [row(4, [0, 1])])              # ... and is predicted again
    assert sim.stats["bytes_h2d"] == b
    plan = sim.visit(1, row(4, [0, 1]))
    assert plan.misses == [] and sim.stats["prefetch_used"] == 2


# ------------------------------------------------------------------------------------------------
# Hand-worked scenarios for the readings the paper leaves open (R8, R10, R11, R12, R25; section 4:
# the strict "next use later than the target", hits locked during phase A).  Every expected slot table, wave list and
# counter below is a LITERAL worked out by hand from DESIGN.md section 4's wording -- the steps are in the comments --
# never a value the simulator produced.  Global expert id g = layer * E + e; tables are slot -> g.
# tests/test_oracle_cache.py::test_every_mutation_of_the_simulator_fails_a_pin keeps them sharp.
# ------------------------------------------------------------------------------------------------
def test_r8_completed_victims_farthest_next_use_first(Sim=CacheSim):
    """R8 first key.  3 layers x 1 expert, 2 slots, no predictions (a visit without a supplied prediction counts as
    'assume used', so an expert's next use is its layer's next visit).
    v0: (0,0) missed -> empty slot 0.  v1: (1,0) missed -> empty slot 1.  v2: (2,0) missed, both residents completed:
    (0,0) is next used at v3, (1,0) at v4 -> the JUST-FINISHED layer 1 is the farthest and goes, although layer 0's
    expert is the least recently used (layer 1's slots are reused for layer 3 as layer 1 completes)."""
    sim = Sim(3, 1, 2, W)
    sim.visit(0, [1]); sim.visit(1, [1])
    assert sim.snapshot() == [0, 1]
    plan = sim.visit(2, [1])
    assert plan.misses == [0] and plan.waves == [(0, 1, True)]
    assert sim.snapshot() == [0, 2]
    plan = sim.visit(3, [1])                       # layer 0 again: still resident
    assert plan.hits == [0] and sim.snapshot() == [0, 2]
    assert sim.stats == dict(lookups=4, hits=1, misses=3, prefetch_issued=0, prefetch_used=0, prefetch_wasted=0,
                             ondemand_loads=3, evictions=1, bytes_h2d=3 * W)


def test_r8_equal_next_use_falls_back_to_least_recently_used(Sim=CacheSim):
    """R8 second key.  One layer, so every completed expert has the same next use (the next visit) and the LRU stamp
    decides; a HIT refreshes the stamp.  v0: 0 -> slot 0, 1 -> slot 1.  v1: 0 hits (now the most recent).  v2: 2 missed
    -> the victim is expert 1 (older use), not expert 0 (older load)."""
    sim = Sim(1, 4, 2, W)
    sim.visit(0, row(4, [0, 1]))
    sim.visit(1, row(4, [0]))
    sim.visit(2, row(4, [2]))
    assert sim.snapshot() == [0, 2]


def test_r11_last_resort_takes_the_prefetch_needed_latest(Sim=CacheSim):
    """R11 (class 3).  3 layers x 2 experts, 2 slots, horizon = fill.  Warm-up prefetch with predicted sets v0: {},
    v1: {0}, v2: {0} loads (1,0) -> slot 0 for v1 and (2,0) -> slot 1 for v2.  At v0 the gate selects (0,0): a miss,
    and the pool holds nothing but prefetches whose visits are still to come (not mis-prefetched, not completed), so
    phase A finds no victim and phase B takes class 3: the one needed LATEST, (2,0) at v2, not (1,0) at v1 -- although
    (1,0) is the older load."""
    sim = Sim(3, 2, 2, W)
    assert sim.prefetch(-1, [row(2, []), row(2, [0]), row(2, [0])]) == 2
    assert sim.snapshot() == [2, 4]
    plan = sim.visit(0, row(2, [0]))
    assert plan.misses == [0] and plan.waves == [(0, 1, True)]
    assert sim.snapshot() == [2, 0]
    assert sim.stats["prefetch_wasted"] == 1 and sim.stats["evictions"] == 1 and sim.stats["ondemand_loads"] == 1
    plan = sim.visit(1, row(2, [0]))               # the prefetch for v1 survived and is used
    assert plan.hits == [0] and sim.stats["prefetch_used"] == 1


def test_prefetch_never_evicts_an_expert_needed_at_the_target_visit(Sim=CacheSim):
    """Class 2 wants a next use strictly LATER than the target.  One layer x 3 experts, 2 slots, H = 1.  v0: {0, 1}
    loaded on demand.  Predicted for v1: {0, 1, 2}: 0 and 1 are resident; for 2 the only candidates are 0 and 1, whose
    next use IS the target visit -> no victim, nothing moves ("the cache is full of useful experts")."""
    sim = Sim(1, 3, 2, W, horizon=1)
    sim.visit(0, row(3, [0, 1]))
    assert sim.prefetch(0, [row(3, [0, 1, 2])]) == 0
    assert sim.snapshot() == [0, 1]
    assert sim.stats["bytes_h2d"] == 2 * W and sim.stats["evictions"] == 0 and sim.stats["prefetch_issued"] == 0


def test_r12_misses_are_served_in_ascending_expert_order(Sim=CacheSim):
    """R12.  (a) two misses, two empty slots: the lower expert id is served first and takes the lower slot.
    (b) one layer x 4 experts, 2 slots holding {0, 1}; v1 selects {0, 2, 3}: 0 hits and is locked; phase A serves 2
    first -> the completed expert 1's slot 1; 3 finds every slot locked and waits for phase B, where both residents
    are completed with the same next use and expert 0 (used at tick 3) is older than expert 2 (loaded at tick 4)
    -> slot 0.  Served in descending order the table would end as [2, 3]."""
    sim = Sim(1, 4, 2, W)
    plan = sim.visit(0, row(4, [2, 3]))
    assert plan.misses == [2, 3] and plan.waves == [(2, 0, True), (3, 1, True)] and sim.snapshot() == [2, 3]
    sim = Sim(1, 4, 2, W)
    sim.visit(0, row(4, [0, 1]))
    plan = sim.visit(1, row(4, [0, 2, 3]))
    assert plan.hits == [0] and plan.misses == [2, 3]
    assert plan.waves == [(0, 0, False), (2, 1, True), (3, 0, True)]
    assert sim.snapshot() == [3, 2]


def test_r12_prefetches_are_issued_in_ascending_expert_order(Sim=CacheSim):
    sim = Sim(2, 4, 4, W)
    assert sim.prefetch(-1, [row(4, [1, 3]), row(4, [0, 2])]) == 4
    assert sim.snapshot() == [1, 3, 4, 6]          # visit order first, then expert id; lowest empty slot each time


def test_r10_horizon_limits_how_far_ahead_prefetch_loads(Sim=CacheSim):
    """R10.  H = 1 with two visits' predictions supplied: only the next visit's expert is loaded; the second row is
    kept as knowledge (it still feeds the next-use estimate)."""
    sim = Sim(2, 2, 4, W, horizon=1)
    assert sim.prefetch(-1, [row(2, [0]), row(2, [1])]) == 1
    assert sim.snapshot() == [0, -1, -1, -1]
    sim = Sim(2, 2, 4, W, horizon=0)
    assert sim.prefetch(-1, [row(2, [0]), row(2, [1])]) == 2
    assert sim.snapshot() == [0, 3, -1, -1]


def test_r25_retargeted_prefetch_is_no_longer_a_misprefetch_victim(Sim=CacheSim):
    """R25.  2 layers x 4 experts, 2 slots, horizon = fill.  Warm-up: predicted v0 = {0, 1}, v1 = {} -> (0,0) -> slot 0,
    (0,1) -> slot 1, both for v0.  v0 selects only (0,0): (0,1) is now a stale prefetch.  After v0 the predictor says
    v1 = {}, v2 = {0, 1}: both are resident, nothing is loaded, and the stale (0,1) is RE-TARGETED to v2.
    v1 selects (1,3), a miss: (0,1) is a prefetch whose visit (v2) is still to come -- not mis-prefetched -- so the victim
    is the completed (0,0) (next use v2 > v1).  Without the re-target (0,1) would count as mis-prefetched (its visit v0 has
    passed) and be the first victim, and prefetch_wasted would be 1."""
    sim = Sim(2, 4, 2, W)
    assert sim.prefetch(-1, [row(4, [0, 1]), row(4, [])]) == 2
    assert sim.snapshot() == [0, 1]
    sim.visit(0, row(4, [0]))
    assert sim.prefetch(0, [row(4, []), row(4, [0, 1])]) == 0
    plan = sim.visit(1, row(4, [3]))
    assert plan.misses == [3] and plan.waves == [(3, 0, True)]
    assert sim.snapshot() == [7, 1]
    assert sim.stats["prefetch_wasted"] == 0 and sim.stats["evictions"] == 1
    plan = sim.visit(2, row(4, [0, 1]))            # the re-targeted prefetch is used; (0,0) has to come back
    assert plan.hits == [1] and plan.misses == [0]
    assert sim.stats["prefetch_used"] == 2 and sim.stats["bytes_h2d"] == 4 * W


def test_next_use_estimate_follows_the_supplied_predictions(Sim=CacheSim):
    """est_next_use: inside the supplied predictions an expert's next use is the first visit of its layer that predicts
    it.  2 layers x 2 experts, 2 slots.  v0: (0,0) -> slot 0; v1: (1,0) -> slot 1.  After v1 the predictor says v2 = {1},
    v3 = {0}.  (0,1) is wanted for v2: (0,0) is NOT predicted at v2, so its next use is v4 (layer 0's following visit, no
    prediction supplied: assume used); (1,0) is predicted at v3.  Both are later than the target v2; the farther one,
    (0,0), goes.  Ignoring the predictions, (0,0) would be 'needed at v2' and (1,0) would be the victim."""
    sim = Sim(2, 2, 2, W)
    sim.visit(0, row(2, [0])); sim.visit(1, row(2, [0]))
    assert sim.snapshot() == [0, 2]
    assert sim.prefetch(1, [row(2, [1]), row(2, [0])]) == 1
    assert sim.snapshot() == [1, 2]
    plan = sim.visit(2, row(2, [1]))
    assert plan.hits == [1] and plan.misses == []


def test_misprefetched_victims_oldest_first(Sim=CacheSim):
    """Class 1 order: among several mis-prefetched experts the one loaded first goes first.  One layer x 4 experts,
    3 slots: {0, 1, 2} prefetched for v0 (slots 0, 1, 2); v0 selects {2, 3}: 2 hits, 3 takes expert 0's slot."""
    sim = Sim(1, 4, 3, W)
    sim.prefetch(-1, [row(4, [0, 1, 2])])
    sim.visit(0, row(4, [2, 3]))
    assert sim.snapshot() == [3, 1, 2]


def test_phase_a_never_destroys_a_still_useful_prefetch(Sim=CacheSim):
    """Phase A takes victims from classes 0-2 only.  2 layers x 3 experts, 2 slots: (0,0) prefetched for v0 (slot 0), (1,0)
    for v1 (slot 1).  v0 selects {0, 1}: 0 hits; for 1 the only unlocked slot holds a prefetch whose visit is still to
    come, so the load WAITS for phase B and then reuses the slot of this visit's completed hit (class 2 beats class 3);
    the prefetch for v1 survives and nothing is wasted."""
    sim = Sim(2, 3, 2, W)
    assert sim.prefetch(-1, [row(3, [0]), row(3, [0])]) == 2
    assert sim.snapshot() == [0, 3]
    plan = sim.visit(0, row(3, [0, 1]))
    assert plan.waves == [(0, 0, False), (1, 0, True)]
    assert sim.snapshot() == [1, 3] and sim.stats["prefetch_wasted"] == 0
    assert sim.visit(1, row(3, [0])).hits == [0]


def test_hits_of_the_visit_are_never_phase_a_victims(Sim=CacheSim):
    """One layer x 3 experts, 2 slots holding {0, 1}; v1 selects {0, 1, 2}: both residents are this visit's hits (locked),
    so 2 waits for phase B and then takes the older hit's slot -- after that hit's wave was enqueued (R9)."""
    sim = Sim(1, 3, 2, W)
    sim.visit(0, row(3, [0, 1]))
    plan = sim.visit(1, row(3, [0, 1, 2]))
    assert plan.waves == [(0, 0, False), (1, 1, False), (2, 0, True)]
    assert sim.snapshot() == [2, 1]


# ------------------------------------------------------------------------------------------------
# baseline policies: LRU over the pool, LRU inside a per-layer share
# ------------------------------------------------------------------------------------------------
def one_hot_counts(E, e):
    c = [0] * E
    c[e] = 1
    return c


def test_lru_matches_the_textbook_reference_string(Sim=CacheSim):
    """The classic page-replacement reference string (20 references, 3 frames): LRU takes 12 faults -- one access
    per visit, so the batch semantics (hits before misses) play no part."""
    ref = [7, 0, 1, 2, 0, 3, 0, 4, 2, 3, 0, 3, 2, 1, 2, 0, 1, 7, 0, 1]
    sim = Sim(1, 8, 3, W, policy="lru")
    for v, e in enumerate(ref):
        sim.visit(v, one_hot_counts(8, e))
    assert sim.stats["misses"] == 12 and sim.stats["hits"] == 8
    assert sim.stats["ondemand_loads"] == 12 and sim.stats["evictions"] == 9       # 3 cold loads evict nothing
    assert sim.stats["bytes_h2d"] == 12 * W and sim.stats["prefetch_issued"] == 0
    assert sorted(sim.snapshot()) == [0, 1, 7]


@pytest.mark.parametrize("policy,L", [("lru", 1), ("lru", 3), ("layer_lru", 3)])
def test_lru_against_an_independent_ordered_dict(policy, L, Sim=CacheSim):
    from collections import OrderedDict
    E, S, n = 12, 6, 400
    g = np.random.default_rng(3)
    seq = g.integers(0, E, size=n)
    sim = Sim(L, E, S, W, policy=policy)
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


def test_lru_batch_visit_never_evicts_its_own_experts_while_others_remain(Sim=CacheSim):
    sim = Sim(1, 8, 4, W, policy="lru")
    sim.visit(0, row(8, [0, 1, 2, 3]))
    plan = sim.visit(1, row(8, [2, 3, 4, 5]))                      # hits 2, 3 are locked: 4, 5 replace 0, 1
    assert plan.hits == [2, 3] and plan.misses == [4, 5]
    assert sorted(sim.snapshot()) == [2, 3, 4, 5]
    plan = sim.visit(2, row(8, [0, 1, 2, 3, 4, 5]))                # more active experts than slots: phase B reuses
    assert sim.stats["lookups"] == sim.stats["hits"] + sim.stats["misses"] == 4 + 4 + 6
    assert len(set(x for x in sim.snapshot())) == 4


def test_plec_beats_both_lru_baselines_on_the_stack_trace(Sim=CacheSim):
    """The paper's claim in kind (Fig. 9): with a predicted path, PLEC's hit ratio is far above on-demand LRU's."""
    cfg = wl.scaled(wl.CONFIGS["stack_decode"], d_model=64, d_ff=128, T=16, n_layers=8, n_slots=16)
    plec = run_trace(cfg, H=1, n_steps=10, Sim=Sim)
    tr = wl.routing_trace(cfg, 10)
    for policy in ("lru", "layer_lru"):
        sim = Sim(cfg.n_layers, cfg.n_experts, cfg.n_slots, W, policy=policy)
        for v in range(10 * cfg.n_layers):
            sim.visit(v, np.bincount(tr.sets[v].ravel(), minlength=cfg.n_experts))
        assert plec.hit_ratio() > sim.hit_ratio() + 0.2, policy


# ------------------------------------------------------------------------------------------------
# clairvoyant reference (Belady MIN) for the policy gap: how far PLEC's and LRU's loads are from the floor
# ------------------------------------------------------------------------------------------------
def test_belady_matches_the_textbook_reference_string():
    """The classic reference string again (see the LRU pin above): the optimal policy takes 9 faults with 3 frames."""
    ref = [7, 0, 1, 2, 0, 3, 0, 4, 2, 3, 0, 3, 2, 1, 2, 0, 1, 7, 0, 1]
    loads = belady_min_loads(1, 8, 3, [[e] for e in ref])
    assert sum(loads) == 9
    assert loads[:4] == [1, 1, 1, 1] and loads[4] == 0


def _min_loads_exhaustive(visits, L, E, S):
    """Fewest loads over ALL eviction choices in the same serving model (inside a visit hits first, then the misses in
    ascending id; a miss may evict any resident): memoised search over (visit, miss index, cache)."""
    from functools import lru_cache
    want = [tuple((v % L) * E + e for e in a) for v, a in enumerate(visits)]

    @lru_cache(maxsize=None)
    def go(v, cache):
        if v == len(want):
            return 0
        misses = tuple(g for g in want[v] if g not in cache)
        return serve(v, misses, cache)

    @lru_cache(maxsize=None)
    def serve(v, misses, cache):
        if not misses:
            return go(v + 1, cache)
        g, rest = misses[0], misses[1:]
        if len(cache) < S:
            return 1 + serve(v, rest, tuple(sorted(cache + (g,))))
        return 1 + min(serve(v, rest, tuple(sorted(tuple(x for x in cache if x != out) + (g,)))) for out in cache)
    return go(0, ())


@pytest.mark.parametrize("seed", range(12))
def test_belady_is_optimal_on_small_traces(seed):
    g = np.random.default_rng(seed)
    L, E, S = int(g.integers(1, 3)), 4, int(g.integers(2, 4))
    visits = [sorted(set(int(e) for e in g.choice(E, size=int(g.integers(1, 4)), replace=False))) for _ in range(10)]
    assert sum(belady_min_loads(L, E, S, visits)) == _min_loads_exhaustive(visits, L, E, S)


def test_policy_gap_to_the_clairvoyant_floor_on_the_decode_traces():
    """Loads per step of PLEC (config horizon), on-demand LRU and the clairvoyant floor on the cfg 3 and (reduced-length)
    cfg 5 routing traces: the floor is never beaten, and the numbers quoted in profiles/r2_policies.md come from here
    (run with -s)."""
    for name, steps, horizons in (("mixtral_decode", 256, (1,)), ("stack_decode", 16, (0, 1))):
        cfg = wl.scaled(wl.CONFIGS[name], d_model=64, d_ff=128)
        tr = wl.routing_trace(cfg, steps)
        L, E = cfg.n_layers, cfg.n_experts
        nv = steps * L
        acts = [sorted(set(int(e) for e in tr.sets[v].ravel())) for v in range(nv)]
        floor = sum(belady_min_loads(L, E, cfg.n_slots, acts)) / steps
        rows = {"clairvoyant (Belady MIN, demand)": floor}
        for H in horizons:
            sim = run_trace(wl.scaled(cfg, horizon=H), H, steps)
            rows[f"PLEC H={'fill' if H <= 0 else H}"] = (sim.stats["ondemand_loads"] + sim.stats["prefetch_issued"]) / steps
        lru = CacheSim(L, E, cfg.n_slots, W, policy="lru")
        for v in range(nv):
            lru.visit(v, np.bincount(tr.sets[v].ravel(), minlength=E))
        rows["on-demand LRU"] = lru.stats["ondemand_loads"] / steps
        print(name, {k: round(v, 2) for k, v in rows.items()})
        assert all(v >= floor - 1e-9 for v in rows.values())
        assert floor > 0


# ------------------------------------------------------------------------------------------------
# The pins above are only worth something if a plausible mistake in the simulator turns one of them red.  This test
# re-runs every scenario test of this file against one-line MUTANTS of oracle/cache_sim.py (source text edited in
# memory, never written back) and demands that each mutant fails at least one of them (DESIGN.md section 2 has the table
# mutant -> failing pin).  One mutant is EQUIVALENT and says so: not stopping a refill at the first expert without a
# victim cannot change anything, because victims for a later target are a subset of those for an earlier one.
# ------------------------------------------------------------------------------------------------
MUTANTS = [
    ("R8: nearest next use evicted first among completed", "key = (2, -nu, self.slot_stamp[s], s)", "key = (2, nu, self.slot_stamp[s], s)"),
    ("R8: most recently used evicted first among completed", "key = (2, -nu, self.slot_stamp[s], s)", "key = (2, -nu, -self.slot_stamp[s], s)"),
    ("R11: nearest next use evicted first in the last resort", "key = (3, -nu, self.slot_stamp[s], s)", "key = (3, nu, self.slot_stamp[s], s)"),
    ("class 2 admits a next use AT the target", "nu > target", "nu >= target"),
    ("R12: misses served in descending order", "for e in plan.misses:", "for e in reversed(plan.misses):"),
    ("R12: prefetches issued in descending order", "for e in sorted(self.pred[t]):", "for e in sorted(self.pred[t], reverse=True):"),
    ("prefetch walks the visits backwards", "for t in range(v_now + 1, hi + 1):", "for t in range(hi, v_now, -1):"),
    ("R25: no re-target", "self.slot_pred_for[s] = t   # R25", "pass   # R25"),
    ("P:L130: mis-prefetched demoted below completed", "key = (1, 0, self.slot_stamp[s], s)", "key = (2.5, 0, self.slot_stamp[s], s)"),
    ("class 1: newest mis-prefetch first", "key = (1, 0, self.slot_stamp[s], s)", "key = (1, 0, -self.slot_stamp[s], s)"),
    ("a prefetch is mis-prefetched only after its visit", "self.slot_pred_for[s] <= v_now:\n                key = (1,", "self.slot_pred_for[s] < v_now:\n                key = (1,"),
    ("hits are not locked during phase A", "self.slot_stamp[s] = self.tick\n            locked.add(gid(e))", "self.slot_stamp[s] = self.tick"),
    ("phase A may take a still-useful prefetch", "self._victim(v, v, allow3=False, locked=locked)", "self._victim(v, v, allow3=True, locked=locked)"),
    ("next-use estimate ignores the predictions", "while v2 in self.pred and e not in self.pred[v2]:", "while False:"),
    ("a hit does not refresh the LRU stamp", "self.tick += 1\n            self.slot_stamp[s] = self.tick\n            locked.add", "locked.add"),
    ("R10: the horizon is ignored", "(min(self.H, n_ahead) if self.H > 0 else n_ahead)", "n_ahead"),
    ("empty slots are not preferred", "key = (0, 0, 0, s)", "key = (9, 0, 0, s)"),
    ("highest empty slot first", "key = (0, 0, 0, s)", "key = (0, 0, 0, -s)"),
    ("a prefetched expert counts as used from the start", "self.slot_used[s] = False\n        self.tick += 1", "self.slot_used[s] = pred_for != -1\n        self.tick += 1"),
]
EQUIVALENT_MUTANTS = [
    ("prefetch does not stop at the first expert without a victim", "return issued               # pool is full", "continue                    # pool is full"),
]


def _mutant(old, new):
    import oracle.cache_sim as cs
    src = open(cs.__file__).read()
    assert src.count(old) == 1, f"mutation site not unique / not found: {old!r}"
    import sys
    import types
    mod = types.ModuleType("oracle_cache_sim_mutant")
    sys.modules[mod.__name__] = mod              # dataclasses looks the defining module up by name
    try:
        exec(compile(src.replace(old, new), cs.__file__ + "<mutant>", "exec"), mod.__dict__)
    finally:
        del sys.modules[mod.__name__]
    return mod.CacheSim


def _scenario_tests():
    import inspect
    out = []
    for name, fn in sorted(globals().items()):
        if name.startswith("test_") and callable(fn) and "Sim" in inspect.signature(fn).parameters:
            others = [p for p in inspect.signature(fn).parameters.values() if p.name != "Sim" and p.default is p.empty]
            if not others:
                out.append((name, fn))
    return out


def _failing_pins(Sim):
    failed = []
    for name, fn in _scenario_tests():
        try:
            fn(Sim=Sim)
        except Exception:            # an assertion, or the mutant running into a dead end
            failed.append(name)
    return failed


def test_the_unmutated_simulator_passes_every_scenario():
    assert len(_scenario_tests()) >= 25
    assert _failing_pins(CacheSim) == []


@pytest.mark.parametrize("what,old,new", MUTANTS, ids=[m[0] for m in MUTANTS])
def test_every_mutation_of_the_simulator_fails_a_pin(what, old, new):
    failed = _failing_pins(_mutant(old, new))
    assert failed, f"mutant survives every pin: {what}"


@pytest.mark.parametrize("what,old,new", EQUIVALENT_MUTANTS, ids=[m[0] for m in EQUIVALENT_MUTANTS])
def test_equivalent_mutants_really_are_equivalent(what, old, new):
    """Stop rule of the refill: after the first expert that finds no class 0-2 victim nothing later in
    the same call can find one -- est_next_use does not depend on the target, a later target only shrinks class 2, no
    stale prefetch is left to re-target (it would have been a class-1 victim) -- so 'stop' and 'skip' are the same
    policy.  Checked on seeded traces, state and log compared after every call."""
    Mut = _mutant(old, new)
    assert _failing_pins(Mut) == []
    for name, H, kw in (("mixtral_decode", 1, {}), ("mixtral_decode", 0, {}), ("stack_decode", 0, dict(T=16, n_layers=6, n_slots=12)),
                        ("stack_decode", 2, dict(T=8, n_layers=5, n_slots=7))):
        cfg = wl.scaled(wl.CONFIGS[name], d_model=64, d_ff=128, **kw)
        a = run_trace(cfg, H, n_steps=40, Sim=CacheSim)
        b = run_trace(cfg, H, n_steps=40, Sim=Mut)
        assert a.log == b.log and a.stats == b.stats and a.snapshot() == b.snapshot()
