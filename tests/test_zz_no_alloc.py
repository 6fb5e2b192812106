"""ef_path_hamming_static (include/ef.h): the no-allocation variant of ef_path_hamming -- its scratch (the bit-packed
paths) is a static device array inside libef.so, resolved with cudaGetSymbolAddress at ef_create, instead of a
cudaMalloc'ed workspace.  Its output must equal the existing path's bit for bit (integer work: the tolerance every
token-scheduler test uses), on two calls in a row that share the array, and it must refuse sizes beyond the array.

This file is collected LAST on purpose (pytest -x: a failure here hides nothing behind it), and it
passes alone in a fresh process as well as after the other tests (it builds its own ctx and its own inputs)."""
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def test_static_scratch_hamming_equals_the_allocating_path_on_two_calls_in_a_row():
    from paper_2410_17954_b200 import EfContext, EfError
    dev = torch.device("cuda", 0)
    ctx = EfContext(n_layers=1, n_experts=8, top_k=2, d_model=256, d_ff=512, n_slots=2, n_shared=0, max_tokens=16)
    try:
        # two problems of different size and word count: several 64 x 64 tiles with a ragged edge and more than one 32-word
        # chunk first, then a smaller one whose packed paths cover only the head of what the first call left in the array
        shapes = [(333, 40, 40, 3), (70, 26, 64, 6)]
        paths = [torch.from_numpy(wl.token_paths(seed=11 + i, n_tokens=N, n_layers=L, n_experts=E, top_k=k, n_families=3,
                                                 family_prob=0.7)).to(dev) for i, (N, L, E, k) in enumerate(shapes)]
        want = [torch.full((p.shape[0], p.shape[0]), 0x7fff, dtype=torch.int16, device=dev) for p in paths]
        got = [torch.full((p.shape[0], p.shape[0]), 0x7ffe, dtype=torch.int16, device=dev) for p in paths]
        for p, d in zip(paths, want):
            ctx.ef_path_hamming(p, d)              # the existing path (allocates its workspace on first use)
        torch.cuda.synchronize()
        free_before, _ = torch.cuda.mem_get_info(dev)
        launches_before = ctx.ef_launch_count()
        for p, d in zip(paths, got):               # two calls in a row on one stream, no synchronisation in between
            ctx.ef_path_hamming_static(p, d)
        torch.cuda.synchronize()
        free_after, _ = torch.cuda.mem_get_info(dev)
        assert ctx.ef_launch_count() - launches_before == 4          # two kernels per call, nothing else
        assert free_after == free_before                             # the calls allocated no device memory
        for p, w, g in zip(paths, want, got):
            assert torch.equal(w, g), p.shape
            assert int(g[0, 0]) == 0 and int(g.view(-1)[1:].max()) > 0     # a real distance matrix, not the fill value
        # a second round over the same array, in the other order
        for p, g in zip(reversed(paths), reversed(got)):
            g.fill_(0x7ffe)
            ctx.ef_path_hamming_static(p, g)
        torch.cuda.synchronize()
        for w, g in zip(want, got):
            assert torch.equal(w, g)
        # beyond the static array: N * ceil(LE / 32) * 4 bytes > EF_STATIC_SCRATCH_BYTES (1 MiB) is refused, nothing runs
        N, LE = 4096, 2048 + 32
        big = torch.zeros((N, LE), dtype=torch.uint8, device=dev)
        out = torch.full((N, N), 0x7ffd, dtype=torch.int16, device=dev)
        launches_before = ctx.ef_launch_count()
        with pytest.raises(EfError) as e:
            ctx.ef_path_hamming_static(big, out)
        assert e.value.code == -6 and "static scratch" in str(e.value)      # EF_ERR_CAPACITY
        assert ctx.ef_launch_count() == launches_before
        torch.cuda.synchronize()
        assert int(out[0, 0]) == 0x7ffd and int(out[-1, -1]) == 0x7ffd
        # exactly at the limit it runs: 4096 x 2048 path entries = 1 MiB of packed paths
        at = torch.zeros((N, 2048), dtype=torch.uint8, device=dev)
        at[1::2, ::3] = 1
        ref = torch.empty((N, N), dtype=torch.int16, device=dev)
        ctx.ef_path_hamming(at, ref)
        ctx.ef_path_hamming_static(at, out)
        torch.cuda.synchronize()
        assert torch.equal(ref, out)
    finally:
        ctx.close()
