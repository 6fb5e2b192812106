"""GPU parity of the Token Scheduler (§3.3) against oracle/token_sched.py, through the C ABI.
Everything here is integer work: distances, assignment, permutation, round count and objectives are bit-exact."""
import json
import os

import numpy as np
import pytest

import workloads as wl
from oracle import token_sched as ots

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def ctx():
    from paper_2410_17954_b200 import EfContext
    c = EfContext(n_layers=1, n_experts=8, top_k=2, d_model=256, d_ff=512, n_slots=2, n_shared=0, max_tokens=16)
    yield c
    c.close()


def run_schedule(ctx, r, c0, c1, max_iter=16):
    dev = torch.device("cuda", 0)
    N = len(r)
    p = torch.from_numpy(np.ascontiguousarray(r, np.uint8)).to(dev)
    batch_of = torch.full((N,), -7, dtype=torch.int32, device=dev)
    perm = torch.full((N,), -7, dtype=torch.int32, device=dev)
    info = torch.full((8,), -7, dtype=torch.int32, device=dev)
    bp = torch.full((2, r[0].size), 9, dtype=torch.uint8, device=dev)
    ctx.ef_token_schedule(p, c0, c1, max_iter, batch_of, perm, info, bp)
    torch.cuda.synchronize()
    return batch_of.cpu().numpy(), perm.cpu().numpy(), info.cpu().numpy(), bp.cpu().numpy()


def check_against_oracle(ctx, r, c0, c1, max_iter=16):
    """Both device paths (single-CTA for N <= 256, multi-kernel) against the oracle."""
    ref = ots.schedule(r, c0, c1, max_iter)
    for force_multi in (False, True):
        ctx.ef_set_option(5, 1 if force_multi else 0)          # EF_OPT_TOKEN_SCHED_PATH
        b, p, info, bp = run_schedule(ctx, r, c0, c1, max_iter)
        assert np.array_equal(b, ref.batch_of), force_multi
        for c in (0, 1):
            assert np.array_equal(bp[c], ots.batch_path(r, np.flatnonzero(ref.batch_of == c))), force_multi
        assert np.array_equal(p, ref.perm), force_multi
        assert info[:6].tolist() == [ref.iters, int(ref.converged), ref.centroids[0], ref.centroids[1], ref.objective,
                                     ref.objective_before], force_multi
    ctx.ef_set_option(5, 0)
    return ref


@pytest.mark.parametrize("N,L,E,k", [(8, 1, 4, 2), (64, 4, 8, 2), (129, 3, 5, 1), (200, 32, 8, 2), (70, 26, 64, 6),
                                     (1, 2, 8, 2), (333, 40, 40, 3)])
def test_hamming_matrix_bit_exact(ctx, N, L, E, k):
    """Eq. 6 distances: several 64 x 64 tiles plus a ragged edge, LE below / equal to / above one 32-word chunk."""
    r = wl.token_paths(seed=N + L, n_tokens=N, n_layers=L, n_experts=E, top_k=k, n_families=3, family_prob=0.7)
    dev = torch.device("cuda", 0)
    d = torch.full((N, N), 0x7fff, dtype=torch.int16, device=dev)
    ctx.ef_path_hamming(torch.from_numpy(r).to(dev), d)
    torch.cuda.synchronize()
    got = d.cpu().numpy().view(np.uint16).astype(np.int64)
    assert np.array_equal(got, ots.hamming_matrix(r))


def test_hamming_arbitrary_bits_not_only_topk(ctx):
    g = np.random.default_rng(2)
    r = (g.random((96, 7, 13)) < 0.3).astype(np.uint8) * 255       # any nonzero byte counts as "on the path"
    dev = torch.device("cuda", 0)
    d = torch.zeros((96, 96), dtype=torch.int16, device=dev)
    ctx.ef_path_hamming(torch.from_numpy(r).to(dev), d)
    torch.cuda.synchronize()
    assert np.array_equal(d.cpu().numpy().view(np.uint16).astype(np.int64), ots.hamming_matrix(r))


def test_fig4_example_on_gpu(ctx):
    gld = json.load(open(os.path.join(GOLD, "token_scheduler_fig4.json")))
    r = np.zeros((8, 1, 4), np.uint8)
    for i, es in enumerate(gld["token_experts"]):
        r[i, 0, es] = 1
    ref = check_against_oracle(ctx, r, *gld["init_centroids"])
    assert ref.objective == gld["expected"]["objective_after"] and ref.objective_before == gld["expected"]["objective_before"]


@pytest.mark.parametrize("N,L,E,k,fam,prob", [
    (2, 1, 4, 1, 2, 1.0), (8, 2, 4, 2, 2, 0.9), (32, 1, 8, 2, 2, 0.8),        # cfg 3: 2 x 16 decode tokens, one layer
    (128, 32, 8, 2, 2, 0.6), (128, 32, 8, 2, 4, 0.5), (256, 32, 8, 2, 3, 0.5), (254, 26, 64, 6, 2, 0.5), (258, 4, 8, 2, 2, 0.5),                      # cfg 5: 2 x 64 tokens, 32 x 8 paths
    (1000, 8, 16, 2, 3, 0.7), (1002, 8, 16, 2, 3, 0.7), (1030, 5, 7, 1, 2, 0.5),   # vector / scalar row paths, ragged tiles
    (2048, 26, 64, 6, 2, 0.5),                                                # many-expert paths: 52 words per token
])
def test_schedule_matches_oracle(ctx, N, L, E, k, fam, prob):
    r = wl.token_paths(seed=17 + N, n_tokens=N, n_layers=L, n_experts=E, top_k=k, n_families=fam, family_prob=prob)
    g = np.random.default_rng(N)
    for _ in range(3):
        c0, c1 = (int(v) for v in g.choice(N, 2, replace=False))
        check_against_oracle(ctx, r, c0, c1)


def test_schedule_full_size_prefill_dual_batch(ctx):
    """Two Mixtral prefill batches of 2048 tokens (BASELINE.json configs[1] shape): N = 4096, L x E = 32 x 8."""
    r = wl.token_paths(seed=99, n_tokens=4096, n_layers=32, n_experts=8, top_k=2, n_families=2, family_prob=0.6)
    ref = check_against_oracle(ctx, r, 5, 4000)
    assert ref.objective <= ref.objective_before


def test_iteration_cap_and_ties(ctx):
    r = wl.token_paths(seed=3, n_tokens=256, n_layers=6, n_experts=8, top_k=2, n_families=5, family_prob=0.4)
    for max_iter in (1, 2, 3, 64):
        check_against_oracle(ctx, r, 10, 200, max_iter)
    same = np.zeros((64, 2, 4), np.uint8)
    same[:, :, 1] = 1                                 # identical paths: every margin ties, split by index
    ref = check_against_oracle(ctx, same, 40, 3)
    assert ref.batch_of.tolist() == [0] * 32 + [1] * 32
    top1 = np.zeros((16, 1, 4), np.uint8)             # top-1 over 4 experts: the two non-centroid experts tie
    top1[np.arange(16), 0, np.arange(16) % 4] = 1
    check_against_oracle(ctx, top1, 0, 1)


def test_repeated_calls_reuse_workspace(ctx):
    for N in (64, 512, 64):
        r = wl.token_paths(seed=N, n_tokens=N, n_layers=4, n_experts=8, top_k=2)
        check_against_oracle(ctx, r, 0, N - 1)


@pytest.mark.parametrize("n_src,n,row_elems,dtype", [(64, 64, 256, "bf16"), (100, 37, 8, "f32"), (5, 9, 4096, "bf16"), (3, 0, 8, "f32")])
def test_reindex_rows(ctx, n_src, n, row_elems, dtype):
    """Reindex: a pure row gather, bit-exact."""
    dev = torch.device("cuda", 0)
    g = np.random.default_rng(n_src + n)
    if dtype == "bf16":
        src = torch.from_numpy(g.integers(0, 1 << 15, (n_src, row_elems)).astype(np.int16)).to(dev)
    else:
        src = torch.from_numpy(g.standard_normal((n_src, row_elems)).astype(np.float32)).to(dev)
    perm_np = g.integers(0, n_src, n).astype(np.int32)
    perm = torch.from_numpy(perm_np).to(dev)
    dst = torch.zeros((max(n, 1), row_elems), dtype=src.dtype, device=dev)
    ctx.ef_reindex_rows(src, perm, dst)
    torch.cuda.synchronize()
    assert np.array_equal(dst.cpu().numpy()[:n], src.cpu().numpy()[perm_np])


def test_bad_arguments_are_codes(ctx):
    from paper_2410_17954_b200.binding import EfError
    dev = torch.device("cuda", 0)
    p = torch.zeros((6, 8), dtype=torch.uint8, device=dev)
    out = [torch.zeros(8, dtype=torch.int32, device=dev) for _ in range(3)]
    for N, c0, c1, it in ((6, 0, 0, 4), (6, 0, 6, 4), (6, -1, 2, 4), (6, 0, 1, 0), (5, 0, 1, 4)):
        with pytest.raises(EfError):
            ctx.ef_token_schedule(p[:N], c0, c1, it, *out)
    with pytest.raises(EfError):
        ctx.ef_token_schedule(p, 0, 1, 65, *out)


# ------------------------------------------------------------------------------------------------
# the scheduler in the path: two incoming batches per step -> schedule -> Reindex -> 2 x L visits (§4.2)
# ------------------------------------------------------------------------------------------------
def test_dual_batch_pipeline_matches_oracle_chain():
    """Reduced dual_batch_stack: assignment, batch paths, slot table and counters bit-exact at every visit; the final
    hidden state of every token within the float bar, in the ORIGINAL token order after undoing the permutation."""
    import oracle
    from oracle.cache_sim import CacheSim
    from paper_2410_17954_b200 import DualBatchRunner
    from test_gpu_layer import assert_cache_equal, build_runner
    from test_gpu_stages import bf, check_float, dev_bf16, to_bits

    cfg = wl.scaled(wl.CONFIGS["dual_batch_stack"], d_model=256, d_ff=512, T=8, n_layers=4, n_slots=10)
    L, E, T, N = cfg.n_layers, cfg.n_experts, cfg.T, 2 * cfg.T
    n_steps = 5
    tr = wl.dual_batch_trace(cfg, n_steps, n_families=2, family_prob=0.85)
    r, ex = build_runner(cfg, horizon=0)
    db = DualBatchRunner(r, max_iter=8)
    sim = CacheSim(L, E, cfg.n_slots, cfg.expert_bytes, 0)
    wrs = [wl.router_weight(cfg, l) for l in range(L)]
    dev = torch.device("cuda", 0)
    g = np.random.default_rng(1)
    improved = 0
    for s in range(n_steps):
        pred_paths = wl.sets_to_paths(tr.pred_sets[s], E)
        bias = wl.bias_from_sets(cfg, tr.sets[s])
        x = wl.normal_bf16(cfg.seed, f"x.dual.step{s}", (N, cfg.d_model), 1.0)
        c0, c1 = (int(v) for v in g.choice(N, 2, replace=False))
        # oracle side: schedule, Reindex, batch-level predicted paths (Eq. 4 with OR)
        sc = ots.schedule(pred_paths, c0, c1, 8)
        rows_ref = np.concatenate([ots.batch_path(pred_paths, sc.perm[b * T:(b + 1) * T]).reshape(L, E) for b in (0, 1)])
        improved += sc.objective < sc.objective_before
        # device side
        rows = db.schedule(torch.from_numpy(pred_paths).to(dev), c0, c1, dev_bf16(x), torch.from_numpy(bias).to(dev))
        assert np.array_equal(db.perm.cpu().numpy(), sc.perm)
        assert np.array_equal(rows, rows_ref)
        assert np.array_equal(to_bits(db.x_re), x[sc.perm])
        v0 = s * 2 * L
        sim.prefetch(v0 - 1, rows_ref)

        def on_visit(v, b, l, dst):
            members = sc.perm[b * T:(b + 1) * T]
            counts = np.bincount(tr.sets[s][members, l].ravel(), minlength=E)
            sim.visit(v, counts)
            nxt = rows_ref[b * L + l + 1:]
            if len(nxt):
                sim.prefetch(v, nxt)
            assert_cache_equal(r, sim)

        out = torch.empty((N, cfg.d_model), dtype=torch.bfloat16, device=dev)
        db.run_step(s, rows, db.x_re, db.bias_re, out, on_visit=on_visit)
        r.ctx.ef_sync()
        got = bf(to_bits(out))
        # oracle chain per token in the ORIGINAL order: the result must not depend on the batching
        ref_all = np.zeros((N, cfg.d_model))
        for b in (0, 1):
            members = np.arange(b * T, (b + 1) * T)
            h = x[members]
            for l in range(L):
                u = oracle.round_bf16(oracle.rmsnorm(h, 1e-5))
                ref = oracle.layer_forward(u, wrs[l], bias[members, l], [ex[(l, e)] for e in range(E)], cfg.top_k, res=h)
                h = oracle.round_bf16(ref.out)
            ref_all[members] = bf(h)
        check_float(got, ref_all[sc.perm])
    assert improved >= 1
    r.close()


def test_dual_batch_overlapped_schedule_equals_sequential():
    """§4.2: scheduling unit n+1 on the side stream while unit n decodes changes nothing -- permutation,
    batch paths, reindexed rows, cache counters and final hidden states equal those of the sequential pipeline."""
    from paper_2410_17954_b200 import DualBatchRunner
    from test_gpu_layer import build_runner
    from test_gpu_stages import dev_bf16, to_bits

    cfg = wl.scaled(wl.CONFIGS["dual_batch_stack"], d_model=256, d_ff=512, T=8, n_layers=3, n_slots=9)
    L, E, T, N = cfg.n_layers, cfg.n_experts, cfg.T, 2 * cfg.T
    n_steps = 6
    tr = wl.dual_batch_trace(cfg, n_steps, n_families=2, family_prob=0.85)
    dev = torch.device("cuda", 0)
    g = np.random.default_rng(5)
    cents = [tuple(int(v) for v in g.choice(N, 2, replace=False)) for _ in range(n_steps)]
    paths = [torch.from_numpy(wl.sets_to_paths(tr.pred_sets[s], E)).to(dev) for s in range(n_steps)]
    biases = [torch.from_numpy(wl.bias_from_sets(cfg, tr.sets[s])).to(dev) for s in range(n_steps)]
    xs = [dev_bf16(wl.normal_bf16(cfg.seed, f"x.dual.step{s}", (N, cfg.d_model), 1.0)) for s in range(n_steps)]

    def run(overlapped):
        r, _ = build_runner(cfg, horizon=0)
        db = DualBatchRunner(r, max_iter=8)
        outs, perms, rows_all = [], [], []
        if overlapped:
            db.schedule_async(paths[0], *cents[0], xs[0], biases[0], 0)
        for s in range(n_steps):
            if overlapped:
                rows = db.wait_schedule(s & 1).copy()
                perms.append(db.perm.cpu().numpy().copy())          # before the next call overwrites it
                if s + 1 < n_steps:
                    db.schedule_async(paths[s + 1], *cents[s + 1], xs[s + 1], biases[s + 1], (s + 1) & 1)
            else:
                rows = db.schedule(paths[s], *cents[s], xs[s], biases[s]).copy()
                perms.append(db.perm.cpu().numpy().copy())
            out = torch.empty((N, cfg.d_model), dtype=torch.bfloat16, device=dev)
            db.run_step(s, rows, db.x_re, db.bias_re, out)
            outs.append(out)
            rows_all.append(rows)
        r.ctx.ef_sync()
        st, snap = r.ctx.ef_cache_get_stats(), r.ctx.ef_cache_snapshot()
        res = [to_bits(o) for o in outs]
        r.close()
        return res, perms, rows_all, st, snap

    a, b = run(False), run(True)
    for s in range(n_steps):
        assert np.array_equal(a[1][s], b[1][s]) and np.array_equal(a[2][s], b[2][s])
        assert np.array_equal(a[0][s], b[0][s])                      # same kernels on the same inputs: same bits
    assert a[3] == b[3] and a[4] == b[4]
