"""Pins for the Token Scheduler oracle (oracle/token_sched.py): what PAPER.md §3.3 and the mathematics fix --
Fig. 4's worked example, Eq. 5 by brute force, Eq. 6 closed forms, the medoid / balance definitions on cases whose
answer is known without running the algorithm.  CPU only."""
import json
import os
from itertools import combinations

import numpy as np
import pytest

import workloads as wl
from oracle import token_sched as ts

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def paths_from_sets(sets, L, E):
    """sets: [N][L][k] expert ids -> binary routing-path matrices r[N, L, E]."""
    r = np.zeros((len(sets), L, E), np.uint8)
    for i, per_layer in enumerate(sets):
        for l, es in enumerate(per_layer):
            for e in es:
                r[i, l, e] = 1
    return r


# ------------------------------------------------------------------------------------------------
# Fig. 4
# ------------------------------------------------------------------------------------------------
def test_fig4_worked_example():
    gld = json.load(open(os.path.join(GOLD, "token_scheduler_fig4.json")))
    L, E, T = gld["n_layers"], gld["n_experts"], gld["tokens_per_batch"]
    exp = gld["expected"]
    r = paths_from_sets([[es] for es in gld["token_experts"]], L, E)
    before = np.repeat([0, 1], T)
    # left of Fig. 4: every original batch engages all experts of the layer; with 2 cached experts that is 2 extra loads
    for b in (0, 1):
        act = int(ts.batch_path(r, np.flatnonzero(before == b)).sum())
        assert act == exp["active_experts_per_original_batch"] == E
        assert act - gld["cache_experts_per_layer"] == exp["extra_loads_per_original_batch"]
    assert ts.objective(r, before) == exp["objective_before"]
    c0, c1 = gld["init_centroids"]
    s = ts.schedule(r, c0, c1)
    assert s.objective_before == exp["objective_before"]
    assert s.objective == exp["objective_after"] == ts.brute_force_optimum(r)
    for b in (0, 1):
        members = np.flatnonzero(s.batch_of == b)
        assert len(members) == T
        bp = ts.batch_path(r, members)
        assert int(bp.sum()) == exp["active_experts_per_scheduled_batch"]
        # "each expert is now assigned more tokens than before"
        per_expert = r.reshape(len(r), -1)[members].sum(axis=0)
        assert set(per_expert[bp == 1]) == {exp["tokens_per_active_expert_after"]}
    assert s.converged


def test_eq4_and_reading_contradicts_fig4_or_reading_matches():
    """R14: with the printed AND of Eq. 4 the left side of Fig. 4 would activate NO expert (no expert is shared by all
    tokens of a batch), contradicting 'engaging all experts within the layer'; OR gives all 4."""
    gld = json.load(open(os.path.join(GOLD, "token_scheduler_fig4.json")))
    r = paths_from_sets([[es] for es in gld["token_experts"]], 1, 4).reshape(8, -1)
    first = r[:4]
    assert int(np.bitwise_and.reduce(first, axis=0).sum()) == 0
    assert int(ts.batch_path(r, range(4)).sum()) == 4


# ------------------------------------------------------------------------------------------------
# Eq. 6: Hamming distance / similarity closed forms
# ------------------------------------------------------------------------------------------------
def test_hamming_closed_form_for_topk_paths():
    """Two top-k paths differ in 2 * (L*k - common) entries: each non-shared (layer, expert) choice flips two bits."""
    L, E, k, N = 5, 8, 2, 24
    g = np.random.default_rng(11)
    sets = [[sorted(g.choice(E, k, replace=False).tolist()) for _ in range(L)] for _ in range(N)]
    r = paths_from_sets(sets, L, E)
    d = ts.hamming_matrix(r)
    for i in range(N):
        for j in range(N):
            common = sum(len(set(sets[i][l]) & set(sets[j][l])) for l in range(L))
            assert d[i, j] == 2 * (L * k - common)
    S = ts.similarity_matrix(r)
    assert np.allclose(np.diag(S), 1.0)                      # d_ii = 0
    assert np.allclose(S, S.T) and S.min() >= 0.0 and S.max() <= 1.0
    assert np.allclose(S, 1.0 - d / (L * E))                 # Eq. 6 with the L x E normaliser
    # complementary paths are at distance L*E (similarity 0)
    a = np.zeros((2, 3, 4), np.uint8)
    a[0, :, :2] = 1
    a[1, :, 2:] = 1
    assert ts.hamming_matrix(a)[0, 1] == 12 and ts.similarity_matrix(a)[0, 1] == 0.0


def test_hamming_is_a_metric_and_matches_bit_loop():
    g = np.random.default_rng(5)
    r = (g.random((10, 3, 7)) < 0.4).astype(np.uint8)
    d = ts.hamming_matrix(r)
    flat = r.reshape(10, -1)
    for i in range(10):
        for j in range(10):
            assert d[i, j] == sum(int(a) ^ int(b) for a, b in zip(flat[i], flat[j]))
            for m in range(10):
                assert d[i, j] <= d[i, m] + d[m, j]


def test_hamming_not_confused_with_overlap_or_transposed_layout():
    """A path and a copy with one layer's expert moved differ by exactly 2, wherever the layer is; paths that only
    share zeros are not 'similar' beyond what Eq. 6 gives."""
    L, E = 4, 6
    base = np.zeros((L, E), np.uint8)
    base[np.arange(L), [0, 1, 2, 3]] = 1
    for l in range(L):
        other = base.copy()
        other[l] = 0
        other[l, 5] = 1
        assert ts.hamming_matrix(np.stack([base, other]))[0, 1] == 2


# ------------------------------------------------------------------------------------------------
# Eq. 5 objective: evaluator and optimum by brute force
# ------------------------------------------------------------------------------------------------
def test_objective_counts_active_experts_per_layer_and_batch():
    # 2 layers x 3 experts; batch 0 = tokens {0,1}, batch 1 = tokens {2,3}
    sets = [[[0], [0]], [[1], [0]], [[2], [2]], [[2], [1]]]
    r = paths_from_sets(sets, 2, 3)
    b = np.array([0, 0, 1, 1])
    # batch 0: layer0 {0,1}, layer1 {0} -> 3; batch 1: layer0 {2}, layer1 {1,2} -> 3
    assert ts.objective(r, b) == 6
    # regrouping tokens {0,2} | {1,3}: layer0 {0,2}, layer1 {0,2} -> 4; layer0 {1,2}, layer1 {0,1} -> 4
    assert ts.objective(r, np.array([0, 1, 0, 1])) == 8


@pytest.mark.parametrize("seed", range(6))
def test_heuristic_never_beats_brute_force_and_is_balanced(seed):
    L, E, k, T = 3, 6, 2, 5
    g = np.random.default_rng(100 + seed)
    sets = [[g.choice(E, k, replace=False).tolist() for _ in range(L)] for _ in range(2 * T)]
    r = paths_from_sets(sets, L, E)
    opt = ts.brute_force_optimum(r)
    # the optimum by an independent enumeration of all balanced splits
    vals = []
    for t1 in combinations(range(2 * T), T):
        b = np.ones(2 * T, int)
        b[list(t1)] = 0
        vals.append(sum(len({(l, e) for i in np.flatnonzero(b == c) for l in range(L) for e in sets[i][l]}) for c in (0, 1)))
    assert opt == min(vals)
    for c0, c1 in ((0, 1), (3, 7), (9, 2)):
        s = ts.schedule(r, c0, c1)
        assert s.objective >= opt
        assert sorted(s.perm.tolist()) == list(range(2 * T))
        assert (s.batch_of == 0).sum() == T == (s.batch_of == 1).sum()
        assert s.perm[:T].tolist() == sorted(np.flatnonzero(s.batch_of == 0).tolist())
        assert s.perm[T:].tolist() == sorted(np.flatnonzero(s.batch_of == 1).tolist())
        assert s.objective == ts.objective(r, s.batch_of)
        assert 1 <= s.iters <= 16


# ------------------------------------------------------------------------------------------------
# K-means steps on cases with a known answer
# ------------------------------------------------------------------------------------------------
def test_medoid_of_a_star_is_its_centre():
    """Centre path p; every other member differs from p in one layer (distance 2) and from each other in two
    layers (distance 4): the centre has the highest average similarity to the others."""
    L, E = 6, 8
    p = np.zeros((L, E), np.uint8)
    p[np.arange(L), 0] = 1
    members = [p]
    for l in range(5):
        q = p.copy()
        q[l] = 0
        q[l, 1 + l] = 1
        members.append(q)
    order = [3, 0, 5, 1, 2, 4]                      # the centre is token 1 after shuffling
    r = np.stack([members[i] for i in order])
    d = ts.hamming_matrix(r)
    assert ts.medoid(d, range(6)) == 1
    # restricted to a sub-cluster without the centre all members tie -> the lowest index wins (R27)
    assert ts.medoid(d, [0, 2, 4, 5]) == 0


def test_assignment_is_top_T_by_margin_with_index_ties():
    # distances to the two centroids given directly: margin = d[i,c1] - d[i,c0]
    n = 6
    d = np.zeros((n, n), np.int64)
    c0, c1 = 0, 5
    to_c0 = [0, 2, 4, 4, 6, 6]
    to_c1 = [6, 4, 4, 4, 2, 0]
    for i in range(n):
        d[i, c0] = d[c0, i] = to_c0[i]
        d[i, c1] = d[c1, i] = to_c1[i]
    # margins: 6, 2, 0, 0, -4, -6 -> cluster 0 = {0, 1} + the lower-index tie (2)
    assert ts.assign_balanced(d, c0, c1).tolist() == [0, 0, 0, 1, 1, 1]
    # an over-full preferred cluster sheds its weakest members: margins 6, 4, 2, 2, 1, -6 -> T = 3 keeps {0, 1, 2}
    to_c1 = [6, 6, 6, 6, 7, 0]
    to_c0 = [0, 2, 4, 4, 6, 6]
    for i in range(n):
        d[i, c0] = d[c0, i] = to_c0[i]
        d[i, c1] = d[c1, i] = to_c1[i]
    assert ts.assign_balanced(d, c0, c1).tolist() == [0, 0, 0, 1, 1, 1]


@pytest.mark.parametrize("c0,c1", [(0, 9), (3, 12), (15, 4)])
def test_two_disjoint_families_are_recovered_exactly(c0, c1):
    """Tokens drawn from two path families that use disjoint expert halves: any start with one centroid per family
    recovers the families in one assignment, and the objective reaches the optimum (each batch activates only its
    family's experts)."""
    L, E, k, T = 4, 8, 2, 8
    g = np.random.default_rng(3)
    fam = np.array([0] * T + [1] * T)
    fam = fam[g.permutation(2 * T)]
    if fam[c0] == fam[c1]:
        c1 = int(np.flatnonzero(fam != fam[c0])[0])
    sets = [[(g.choice(4, k, replace=False) + 4 * fam[i]).tolist() for _ in range(L)] for i in range(2 * T)]
    r = paths_from_sets(sets, L, E)
    s = ts.schedule(r, c0, c1)
    same = (s.batch_of == fam).all() or (s.batch_of == 1 - fam).all()
    assert same and s.converged
    union = [int(ts.batch_path(r, np.flatnonzero(fam == f)).sum()) for f in (0, 1)]
    assert s.objective == sum(union) <= s.objective_before


def test_identical_tokens_split_by_index_and_converge_at_once():
    r = np.zeros((8, 2, 4), np.uint8)
    r[:, :, 1] = 1
    s = ts.schedule(r, 6, 2)
    assert s.batch_of.tolist() == [0, 0, 0, 0, 1, 1, 1, 1]
    assert s.centroids == (0, 4) and s.objective == s.objective_before == 4
    assert s.iters == 2 and s.converged          # round 1 moves the centroids to (0, 4), round 2 confirms them


def test_iteration_limit_is_respected():
    g = np.random.default_rng(9)
    r = (g.random((40, 4, 8)) < 0.25).astype(np.uint8)
    s1 = ts.schedule(r, 0, 1, max_iter=1)
    assert s1.iters == 1
    full = ts.schedule(r, 0, 1, max_iter=50)
    assert full.converged and full.iters < 50
    again = ts.schedule(r, 0, 1, max_iter=full.iters)
    assert again.batch_of.tolist() == full.batch_of.tolist()


def test_generated_token_paths_have_topk_ones_per_layer():
    r = wl.token_paths(seed=7, n_tokens=64, n_layers=4, n_experts=8, top_k=2, n_families=2, family_prob=0.8)
    assert r.shape == (64, 4, 8) and r.dtype == np.uint8
    assert (r.sum(axis=2) == 2).all()
    assert np.array_equal(r, wl.token_paths(seed=7, n_tokens=64, n_layers=4, n_experts=8, top_k=2, n_families=2, family_prob=0.8))


def test_scheduled_batches_need_fewer_loads_in_the_cache_simulator():
    """The paper's claim for the scheduler ('reduces I/O overhead by decreasing expert loads'), checked on
    the policy simulator: a perfect predictor, two families, 2 x 8 tokens through a 6-layer stack."""
    from oracle.cache_sim import CacheSim
    cfg = wl.scaled(wl.CONFIGS["dual_batch_stack"], T=8, n_layers=6, n_slots=12, pred_acc=1.0)
    L, E, T = cfg.n_layers, cfg.n_experts, cfg.T
    tr = wl.dual_batch_trace(cfg, 12, n_families=2, family_prob=0.9)
    loads, active = {}, {}
    for sched in (False, True):
        sim = CacheSim(L, E, cfg.n_slots, 1000, 0)
        n_active = 0
        for s in range(12):
            paths = wl.sets_to_paths(tr.pred_sets[s], E)
            perm = ts.schedule(paths, 0, 2 * T - 1, 8).perm if sched else np.arange(2 * T)
            rows = np.concatenate([ts.batch_path(paths, perm[b * T:(b + 1) * T]).reshape(L, E) for b in (0, 1)])
            v0 = s * 2 * L
            sim.prefetch(v0 - 1, rows)
            for b in (0, 1):
                for l in range(L):
                    v = v0 + b * L + l
                    counts = np.bincount(tr.sets[s][perm[b * T:(b + 1) * T], l].ravel(), minlength=E)
                    n_active += int((counts > 0).sum())
                    sim.visit(v, counts)
                    if len(rows[b * L + l + 1:]):
                        sim.prefetch(v, rows[b * L + l + 1:])
        loads[sched] = sim.stats["ondemand_loads"] + sim.stats["prefetch_issued"]
        active[sched] = n_active
        assert sim.stats["misses"] == 0                      # perfect prediction, pool >= two visits' active sets
    assert active[True] < active[False]
    assert loads[True] < loads[False]


# ------------------------------------------------------------------------------------------------
# Eq. 7: batch-level accuracy of a predicted routing path
# ------------------------------------------------------------------------------------------------
def test_batch_accuracy_hand_counted_and_special_cases():
    R = np.array([[1, 1, 0, 0], [0, 1, 1, 1]], np.uint8)          # true: 2 and 3 active experts
    Rh = np.array([[1, 0, 1, 0], [0, 1, 1, 0]], np.uint8)         # predicted: hits 1 of 2 and 2 of 3
    assert ts.batch_accuracy(R, Rh) == pytest.approx((1 / 2 + 2 / 3) / 2)
    assert ts.batch_accuracy(R, R) == 1.0                          # a perfect prediction
    assert ts.batch_accuracy(R, np.ones_like(R)) == 1.0            # Eq. 7 is a recall: over-prediction is not penalised
    assert ts.batch_accuracy(R, np.zeros_like(R)) == 0.0
    assert ts.batch_accuracy(R, 1 - R) == 0.0                      # the complement never hits
    # not symmetric: swapping the roles divides by the predicted counts instead
    assert ts.batch_accuracy(Rh, R) == pytest.approx((1 / 2 + 2 / 2) / 2)


def test_batch_accuracy_is_the_mean_of_per_layer_recalls_vectorised():
    g = np.random.default_rng(11)
    R = (g.random((7, 16)) < 0.4).astype(np.uint8)
    R[:, 0] = 1                                                    # every layer activates something
    Rh = (g.random((7, 16)) < 0.5).astype(np.uint8)
    want = np.mean((R & Rh).sum(1) / R.sum(1))
    assert ts.batch_accuracy(R, Rh) == pytest.approx(want, rel=1e-12)


def test_synthetic_traces_sit_in_the_papers_accuracy_range():
    """the R17 error model at p = 0.85 / 0.8 gives batch-level accuracies like Table 1's
    (73-87 %) or above -- the synthetic predicted paths are no easier than a plausible predictor's."""
    import workloads as wl
    for name, lo in (("mixtral_decode", 0.85), ("stack_decode", 0.95)):
        cfg = wl.CONFIGS[name]
        L = cfg.n_layers
        tr = wl.routing_trace(cfg, 8)
        accs = []
        for s in range(8):
            true = np.zeros((L, cfg.n_experts), np.uint8)
            for l in range(L):
                true[l, np.unique(tr.sets[s * L + l])] = 1
            accs.append(ts.batch_accuracy(true, tr.predicted[s * L:(s + 1) * L]))
        assert lo <= np.mean(accs) <= 1.0, (name, np.mean(accs))
