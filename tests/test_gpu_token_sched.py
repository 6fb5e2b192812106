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
    ctx.ef_token_schedule(p, c0, c1, max_iter, batch_of, perm, info)
    torch.cuda.synchronize()
    return batch_of.cpu().numpy(), perm.cpu().numpy(), info.cpu().numpy()


def check_against_oracle(ctx, r, c0, c1, max_iter=16):
    """Both device paths (single-CTA for N <= 256, multi-kernel) against the oracle."""
    ref = ots.schedule(r, c0, c1, max_iter)
    for force_multi in (False, True):
        ctx.ef_set_token_sched_path(force_multi)
        b, p, info = run_schedule(ctx, r, c0, c1, max_iter)
        assert np.array_equal(b, ref.batch_of), force_multi
        assert np.array_equal(p, ref.perm), force_multi
        assert info[:6].tolist() == [ref.iters, int(ref.converged), ref.centroids[0], ref.centroids[1], ref.objective,
                                     ref.objective_before], force_multi
    ctx.ef_set_token_sched_path(False)
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
