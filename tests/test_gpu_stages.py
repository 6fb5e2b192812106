"""GPU parity, stage by stage ("teacher-forced": each CUDA stage gets the ORACLE's output of the stage
before it as input).  Everything goes through the C ABI (paper_2410_17954_b200.binding).

Bars (BASELINE.json north_star):
  integer / index outputs bit-exact;
  float outputs: max|gpu-ref| <= 2e-2 * max|ref|  and  sum|gpu-ref| / sum|ref| <= 5e-3.
"""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def dev_bf16(bits):
    from paper_2410_17954_b200.layer import bf16_tensor_from_bits
    return bf16_tensor_from_bits(bits, torch.device("cuda", 0))


def to_bits(t):
    from paper_2410_17954_b200.layer import bits_from_bf16_tensor
    return bits_from_bf16_tensor(t)


def bf(bits):
    return wl.bf16_bits_to_f32(bits).astype(np.float64)


def check_float(gpu, ref, max_tol=2e-2, mean_tol=5e-3):
    gpu = np.asarray(gpu, np.float64); ref = np.asarray(ref, np.float64)
    assert gpu.shape == ref.shape
    scale = np.abs(ref).max()
    max_err = np.abs(gpu - ref).max()
    mean_rel = np.abs(gpu - ref).sum() / max(np.abs(ref).sum(), 1e-300)
    assert max_err <= max_tol * scale, f"max abs err {max_err:.3e} > {max_tol} * {scale:.3e}"
    assert mean_rel <= mean_tol, f"mean rel err {mean_rel:.3e} > {mean_tol}"
    return max_err / max(scale, 1e-300), mean_rel


def make_ctx(**kw):
    from paper_2410_17954_b200 import EfContext
    base = dict(n_layers=1, n_experts=8, top_k=2, d_model=256, d_ff=512, n_slots=4, n_shared=0, max_tokens=64)
    base.update(kw)
    return EfContext(**base)


# ------------------------------------------------------------------------------------------------
# a1 router
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T,d,E,k,renorm,bias_kind", [
    (64, 256, 8, 2, 1, "none"), (64, 256, 8, 2, 0, "expert"), (33, 2048, 64, 6, 1, "expert"),
    (16, 4096, 8, 2, 1, "token"), (5, 64, 256, 8, 1, "none"), (1, 128, 3, 1, 0, "none"), (257, 512, 40, 8, 0, "token"),
])
def test_route_topk(T, d, E, k, renorm, bias_kind):
    ctx = make_ctx(n_experts=E, top_k=k, d_model=d, d_ff=128, max_tokens=T)
    x = wl.normal_bf16(11, "x", (T, d), 1.0); wr = wl.normal_bf16(11, "wr", (E, d), 1 / np.sqrt(d))
    bias = None
    if bias_kind == "expert":
        bias = wl.normal_f32(11, "b", (E,), 0.5)
    if bias_kind == "token":
        bias = wl.normal_f32(11, "bt", (T, E), 0.5)
    logits = oracle.router_logits(x, wr, bias)
    idx_ref, w_ref = oracle.topk_gate(logits, k, renorm)

    dx, dwr = dev_bf16(x), dev_bf16(wr)
    db = None if bias is None else torch.from_numpy(bias).cuda()
    idx = torch.empty((T, k), dtype=torch.int32, device="cuda"); w = torch.empty((T, k), device="cuda")
    lg = torch.empty((T, E), device="cuda")
    ctx.ef_route_topk(dx, dwr, db, T, renorm, idx, w, lg)
    torch.cuda.synchronize()
    lg = lg.cpu().numpy().astype(np.float64); idx = idx.cpu().numpy(); w = w.cpu().numpy().astype(np.float64)
    assert np.abs(lg - logits).max() < 2e-5 * max(1.0, np.abs(logits).max())
    # selection: bit-exact wherever the k/(k+1) gap exceeds what fp32 accumulation can move; elsewhere valid
    srt = np.sort(logits, axis=1)[:, ::-1]
    gap = srt[:, k - 1] - srt[:, k] if k < E else np.full(T, np.inf)
    inner = np.min(-np.diff(srt[:, :k], axis=1), axis=1) if k > 1 else np.full(T, np.inf)
    clear = (gap > 1e-4) & (inner > 1e-4)
    assert clear.mean() > 0.95
    assert np.array_equal(idx[clear], idx_ref[clear])
    for t in np.where(~clear)[0]:
        assert len(set(idx[t])) == k
        assert np.all(logits[t, idx[t]] >= srt[t, k - 1] - 1e-4)
    np.testing.assert_allclose(w[clear], w_ref[clear], rtol=2e-4, atol=1e-6)
    # top-k on identical logits: the oracle's selection applied to the fp32 logits the GPU itself produced
    idx_same, _ = oracle.topk_gate(lg, k, renorm)
    assert np.array_equal(idx, idx_same)
    ctx.close()


def test_route_exact_ties_lower_index():
    T, d, E, k = 4, 64, 8, 3
    ctx = make_ctx(n_experts=E, top_k=k, d_model=d, d_ff=128, max_tokens=T)
    x = np.zeros((T, d), np.uint16); wr = np.zeros((E, d), np.uint16)   # all logits = bias
    bias = np.array([[1, 1, 1, 1, 1, 1, 1, 1], [0, 2, 2, 0, 2, 0, 0, 0], [3, 0, 0, 0, 0, 0, 0, 3],
                     [0, 0, 0, 0, 0, 0, 5, 5]], np.float32)
    idx = torch.empty((T, k), dtype=torch.int32, device="cuda"); w = torch.empty((T, k), device="cuda")
    ctx.ef_route_topk(dev_bf16(x), dev_bf16(wr), torch.from_numpy(bias).cuda(), T, 1, idx, w, None)
    ref, wref = oracle.topk_gate(bias.astype(np.float64), k, 1)
    assert np.array_equal(idx.cpu().numpy(), ref)
    np.testing.assert_allclose(w.cpu().numpy(), wref, rtol=1e-6)
    ctx.close()


# ------------------------------------------------------------------------------------------------
# a2 permute
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T,k,E,d", [(64, 2, 8, 256), (0, 2, 8, 64), (1, 1, 1, 64), (4096, 6, 64, 128),
                                     (1000, 8, 256, 64), (37, 3, 5, 192), (2048, 2, 8, 512)])
def test_permute_bit_exact(T, k, E, d):
    ctx = make_ctx(n_experts=E, top_k=k, d_model=d, d_ff=128, max_tokens=max(T, 1))
    g = wl.stream(12, f"perm{T}.{k}.{E}")
    if T > 0:
        # skewed popularity so that some experts are empty and some are huge
        p = np.exp(2.0 * g.standard_normal(E)); p /= p.sum()
        idx = np.stack([g.choice(E, size=k, replace=False, p=p) for _ in range(T)]).astype(np.int32)
    else:
        idx = np.zeros((0, k), np.int32)
    x = wl.normal_bf16(12, "x", (max(T, 1), d), 1.0)[:T]
    counts_r, offsets_r, src_r, inv_r = oracle.permute(idx, E)
    xp_r = oracle.gather_rows(x, src_r, k) if T else np.zeros((0, d), np.uint16)

    R = T * k
    didx = torch.from_numpy(idx).cuda() if T else torch.empty((0, k), dtype=torch.int32, device="cuda")
    dx = dev_bf16(x) if T else torch.empty((0, d), dtype=torch.bfloat16, device="cuda")
    xp = torch.zeros((max(R, 1), d), dtype=torch.bfloat16, device="cuda")
    counts = torch.full((E,), -1, dtype=torch.int32, device="cuda")
    offsets = torch.full((E + 1,), -1, dtype=torch.int32, device="cuda")
    src = torch.full((max(R, 1),), -1, dtype=torch.int32, device="cuda")
    inv = torch.full((max(R, 1),), -1, dtype=torch.int32, device="cuda")
    chost = torch.full((E,), -1, dtype=torch.int32).pin_memory()
    ctx.ef_permute(didx, dx, T, xp, counts, offsets, src, inv, chost)
    torch.cuda.synchronize()
    assert np.array_equal(counts.cpu().numpy(), counts_r)
    assert np.array_equal(chost.numpy(), counts_r)
    assert np.array_equal(offsets.cpu().numpy(), offsets_r)
    assert np.array_equal(src.cpu().numpy()[:R], src_r)
    assert np.array_equal(inv.cpu().numpy()[:R], inv_r)
    assert np.array_equal(to_bits(xp)[:R], xp_r)
    ctx.close()


# ------------------------------------------------------------------------------------------------
# a4 grouped FFN (resident experts)
# ------------------------------------------------------------------------------------------------
def run_resident_ffn(ctx, E, d, f, counts, seed, simt, splitk=0, expert_kind="swiglu", fused=True):
    """Load experts 0..E-1 into slots via the cache, run the grouped FFN on oracle-permuted rows."""
    cfg = wl.scaled(wl.CONFIGS["tiny"], d_model=d, d_ff=f, n_experts=E, seed=seed, expert_kind=expert_kind)
    experts = [wl.expert_weights(cfg, 0, e) for e in range(E)]
    if not getattr(ctx, "_experts_loaded", False):       # repeated calls on one ctx reuse the resident experts
        for e in range(E):
            ctx.ef_host_expert_register(0, e, *experts[e])
        ctx.ef_cache_prefetch(-1, np.ones((1, E), np.uint8))
        ctx._experts_loaded = True
    snap = ctx.ef_cache_snapshot()
    slot_of = {g: s for s, g in enumerate(snap) if g >= 0}
    assert len(slot_of) == E
    R = int(np.sum(counts))
    x_perm = wl.normal_bf16(seed, "xperm", (R, d), 1.0)
    offs = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    y = torch.full((R, d), float("nan"), dtype=torch.bfloat16, device="cuda")
    from paper_2410_17954_b200 import EF_OPT_FUSED_WAVES, EF_OPT_SPLITK
    if simt:
        ctx.ef_diag_set_simt_ffn(True)       # the plain-FMA bring-up backend exists in the diag library only
    ctx.ef_set_option(EF_OPT_SPLITK, splitk)
    ctx.ef_set_option(EF_OPT_FUSED_WAVES, 1 if fused else 0)
    act = [e for e in range(E) if counts[e] > 0]
    ctx.ef_expert_ffn_grouped_resident(dev_bf16(x_perm), [offs[e] for e in act], [counts[e] for e in act],
                                       [slot_of[e] for e in act], y)
    ctx.ef_sync()
    ref = np.zeros((R, d))
    for e in act:
        ref[offs[e]:offs[e + 1]] = oracle.expert_ffn(x_perm[offs[e]:offs[e + 1]], *experts[e])
    return bf(to_bits(y)), ref


FFN_CASES = [
    # E, d, f, counts  (ragged: empty groups, 1-row groups, >128, >256, exact multiples)
    (4, 256, 512, [40, 0, 1, 87]),
    (3, 128, 256, [128, 256, 129]),
    (5, 512, 1408 - 1408 % 128, [300, 7, 0, 513, 64]),
    (2, 64, 128, [1, 1]),
    (2, 1024, 384, [257, 255]),
    # long K loop on one GEMM, short on the other, long on both (balanced tiles: 593 -> 208 + 208 + 177, 300 -> 160 + 140,
    # 513 -> 176 + 176 + 161, 257 -> 144 + 113; both GEMMs of a wave share ONE token tiling)
    (2, 3072, 256, [300, 593]),
    (3, 256, 3072, [513, 257, 130]),
    (2, 3072, 3072, [593, 300]),
    # odd numbers of weight tiles on both GEMMs (f / 128 = 3, d / 256 = 3): the last pair's partner has no weight tile
    (3, 768, 384, [260, 90, 3]),
]

# variant ids: simt = the diag library's plain-FMA backend; splitk 0 = automatic tail split-K (these launches have fewer
# tiles than SMs, so it engages), 1 = off, 2 / 3 / 5 = every tile split into that many K parts (uneven k-block ranges,
# partial-sum workspace, last-arriver reduction); fused = one launch runs both GEMMs (GEMM2 units wait for their token
# tile's h columns), else two launches
FFN_VARIANTS = [(True, 0, True), (False, 1, True), (False, 0, True), (False, 2, True), (False, 3, True), (False, 5, True),
                (False, 0, False), (False, 3, False)]
FFN_VARIANT_IDS = ["simt_debug", "tcgen05_nosplit", "tcgen05_auto", "tcgen05_split2", "tcgen05_split3", "tcgen05_split5",
                   "two_launches_auto", "two_launches_split3"]


@pytest.mark.parametrize("simt,splitk,fused", FFN_VARIANTS, ids=FFN_VARIANT_IDS)
@pytest.mark.parametrize("E,d,f,counts", FFN_CASES)
def test_ffn_grouped_resident(E, d, f, counts, simt, splitk, fused):
    ctx = make_ctx(n_experts=E, top_k=1, d_model=d, d_ff=f, n_slots=E, max_tokens=int(np.sum(counts)), diag=simt)
    got, ref = run_resident_ffn(ctx, E, d, f, counts, seed=13, simt=simt, splitk=splitk, fused=fused)
    assert not np.isnan(got).any()          # every routed row was written
    check_float(got, ref)
    ctx.close()


# Switch-style non-gated ReLU experts (expert_kind = 1, R30): W1 tiles of 256 rows (f = 384: a ragged last
# weight tile, an odd tile count for the CTA pair), all kernel variants
@pytest.mark.parametrize("simt,splitk,fused", [(True, 0, True), (False, 1, True), (False, 0, True), (False, 3, True), (False, 0, False)],
                         ids=["simt_debug", "tcgen05_nosplit", "tcgen05_auto", "tcgen05_split3", "two_launches_auto"])
@pytest.mark.parametrize("E,d,f,counts", [(4, 256, 512, [40, 0, 1, 87]), (3, 768, 3072, [300, 129, 16]),
                                          (2, 1024, 384, [257, 255]), (2, 64, 128, [1, 1])])
def test_ffn_grouped_resident_relu_experts(E, d, f, counts, simt, splitk, fused):
    ctx = make_ctx(n_experts=E, top_k=1, d_model=d, d_ff=f, n_slots=E, max_tokens=int(np.sum(counts)), expert_kind=1, diag=simt)
    got, ref = run_resident_ffn(ctx, E, d, f, counts, seed=29, simt=simt, splitk=splitk, expert_kind="relu", fused=fused)
    assert not np.isnan(got).any()
    check_float(got, ref)
    ctx.close()


def test_ffn_many_groups_many_waves_in_one_launch():
    """64 groups of ragged sizes in ONE launch (the many-expert shape, reduced): more GEMM1 units than CTA pairs, so GEMM2
    units of the early groups run while GEMM1 units of the late groups are still in flight, and every token tile's
    ready counter is exercised; repeated launches re-arm the counters."""
    E, d, f = 64, 256, 384
    g = wl.stream(5, "ffn.many")
    counts = [int(c) for c in g.integers(0, 300, size=E)]
    counts[3], counts[17], counts[40] = 0, 700, 1
    ctx = make_ctx(n_experts=E, top_k=1, d_model=d, d_ff=f, n_slots=E, max_tokens=int(np.sum(counts)))
    for rep in range(3):
        got, ref = run_resident_ffn(ctx, E, d, f, counts, seed=31, simt=False)
        assert not np.isnan(got).any()
        check_float(got, ref)
    ctx.close()


def test_fused_wave_is_bit_identical_to_two_launches_and_to_itself():
    """Race detector for the in-launch GEMM1 -> GEMM2 hand-over (per-token-tile ready counters, generic-proxy stores read
    back through TMA): both modes use the same tiling and the same split-K plan, so ONE launch must give bit for bit what
    two launches give, on every repetition, for ragged random waves that mix empty, tiny, 129..256-row and multi-tile
    groups (more units than CTA pairs, so GEMM2 units of early groups run while late GEMM1 units are in flight)."""
    from paper_2410_17954_b200 import EF_OPT_FUSED_WAVES
    E, d, f = 24, 512, 768
    g = wl.stream(9, "ffn.fused")
    ctx = make_ctx(n_experts=E, top_k=1, d_model=d, d_ff=f, n_slots=E, max_tokens=6000)
    cfg = wl.scaled(wl.CONFIGS["tiny"], d_model=d, d_ff=f, n_experts=E, seed=41)
    for e in range(E):
        ctx.ef_host_expert_register(0, e, *wl.expert_weights(cfg, 0, e))
    ctx.ef_cache_prefetch(-1, np.ones((1, E), np.uint8))
    slot_of = {gid: s for s, gid in enumerate(ctx.ef_cache_snapshot())}
    for trial in range(10):
        kind = g.integers(0, 4, size=E)
        counts = np.where(kind == 0, 0, np.where(kind == 1, g.integers(1, 40, size=E),
                          np.where(kind == 2, g.integers(129, 257, size=E), g.integers(257, 700, size=E)))).astype(int)
        if counts.sum() == 0:
            counts[0] = 5
        offs = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
        R = int(offs[-1])
        x = dev_bf16(wl.normal_bf16(100 + trial, "xperm", (R, d), 1.0))
        act = [e for e in range(E) if counts[e] > 0]
        args = ([int(offs[e]) for e in act], [int(counts[e]) for e in act], [slot_of[e] for e in act])
        outs = []
        for fused in (1, 0, 1, 1):
            y = torch.full((R, d), float("nan"), dtype=torch.bfloat16, device="cuda")
            ctx.ef_set_option(EF_OPT_FUSED_WAVES, fused)
            ctx.ef_expert_ffn_grouped_resident(x, *args, y)
            ctx.ef_sync()
            outs.append(to_bits(y))
        assert not np.isnan(bf(outs[0])).any()
        for o in outs[1:]:
            assert np.array_equal(o, outs[0]), (trial, counts.tolist())
    ctx.close()


def test_ffn_splitk_repeated_launches_rearm_counters():
    """The arrival counters and scheduler words re-arm themselves: many launches in a row, alternating split
    factors, all give the same answer as the unsplit kernel up to fp32 summation order."""
    E, d, f, counts = 3, 512, 1024, [300, 17, 129]
    ctx = make_ctx(n_experts=E, top_k=1, d_model=d, d_ff=f, n_slots=E, max_tokens=int(np.sum(counts)))
    base, ref = run_resident_ffn(ctx, E, d, f, counts, seed=21, simt=False, splitk=1)
    check_float(base, ref)
    for i, mode in enumerate([0, 4, 2, 0, 7, 16, 3, 0]):
        got, _ = run_resident_ffn(ctx, E, d, f, counts, seed=21, simt=False, splitk=mode)
        assert not np.isnan(got).any()
        check_float(got, ref)
        assert np.abs(got - base).max() <= 2e-2 * np.abs(ref).max(), (i, mode)
    ctx.close()


def test_ffn_does_not_touch_rows_outside_groups():
    E, d, f = 2, 128, 256
    counts = [100, 60]
    ctx = make_ctx(n_experts=E, top_k=1, d_model=d, d_ff=f, n_slots=E, max_tokens=400)
    cfg = wl.scaled(wl.CONFIGS["tiny"], d_model=d, d_ff=f, n_experts=E, seed=14)
    for e in range(E):
        ctx.ef_host_expert_register(0, e, *wl.expert_weights(cfg, 0, e))
    ctx.ef_cache_prefetch(-1, np.ones((1, E), np.uint8))
    slot_of = {g: s for s, g in enumerate(ctx.ef_cache_snapshot()) if g >= 0}
    x = dev_bf16(wl.normal_bf16(14, "x", (400, d), 1.0))
    y = torch.full((400, d), 7.0, dtype=torch.bfloat16, device="cuda")
    # groups placed with gaps: rows [10,110) and [200,260)
    ctx.ef_expert_ffn_grouped_resident(x, [10, 200], counts, [slot_of[0], slot_of[1]], y)
    ctx.ef_sync()
    yb = bf(to_bits(y))
    mask = np.ones(400, bool); mask[10:110] = False; mask[200:260] = False
    assert np.all(yb[mask] == 7.0)
    assert not np.any(np.all(yb[~mask] == 7.0, axis=1))
    ctx.close()


# ------------------------------------------------------------------------------------------------
# a5 combine, a8 rmsnorm
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T,k,d,n_shared,with_res", [(64, 2, 256, 0, False), (33, 6, 2048, 2, False),
                                                     (16, 2, 4096, 0, True), (1, 1, 64, 1, True), (0, 2, 64, 0, False)])
def test_combine(T, k, d, n_shared, with_res):
    E = 8
    ctx = make_ctx(n_experts=E, top_k=k, d_model=d, d_ff=128, n_shared=n_shared, max_tokens=max(T, 1))
    g = wl.stream(15, f"comb{T}.{k}")
    R = T * k
    y_perm = wl.normal_bf16(15, "y", (max(R, 1), d), 1.0)[:R]
    inv = g.permutation(R).astype(np.int32)
    w = g.random((T, k)).astype(np.float32)
    res = wl.normal_bf16(15, "res", (max(T, 1), d), 1.0)[:T] if with_res else None
    ysh = wl.normal_bf16(15, "ysh", (max(n_shared * T, 1), d), 1.0)[:n_shared * T] if n_shared else None
    ysh_sum = None if ysh is None else bf(ysh).reshape(n_shared, T, d).sum(0)
    ref = oracle.combine(bf(y_perm), inv, w.astype(np.float64), k, res=res, y_shared=ysh_sum)
    out = torch.zeros((max(T, 1), d), dtype=torch.bfloat16, device="cuda")
    if T:
        ctx.ef_combine(dev_bf16(y_perm), torch.from_numpy(inv).cuda(), torch.from_numpy(w).cuda(), T,
                       None if res is None else dev_bf16(res), None if ysh is None else dev_bf16(ysh), out)
    else:
        ctx.ef_combine(None, None, None, 0, None, None, out)
    torch.cuda.synchronize()
    if T:
        got = bf(to_bits(out))[:T]
        # one bf16 rounding of an fp32 sum: half an ulp relative
        assert np.all(np.abs(got - ref) <= np.abs(ref) * 2.0 ** -8 + 1e-6)
    ctx.close()


@pytest.mark.parametrize("T,d", [(16, 4096), (3, 64), (5, 8192 + 64)])
def test_rmsnorm(T, d):
    ctx = make_ctx(d_model=d, d_ff=128, max_tokens=T)
    x = wl.normal_bf16(16, "x", (T, d), 3.0)
    ref = oracle.rmsnorm(x, 1e-5)
    out = torch.empty((T, d), dtype=torch.bfloat16, device="cuda")
    ctx.ef_rmsnorm(dev_bf16(x), T, 1e-5, out)
    torch.cuda.synchronize()
    got = bf(to_bits(out))
    assert np.all(np.abs(got - ref) <= np.abs(ref) * 2.0 ** -8 + 1e-6)
    ctx.close()


# ------------------------------------------------------------------------------------------------
# error behaviour
# ------------------------------------------------------------------------------------------------
def test_errors_are_codes_not_crashes():
    from paper_2410_17954_b200 import EfContext, EfError
    with pytest.raises(EfError) as e:
        EfContext(1, 8, 2, 100, 512, 4)                 # d_model % 64 != 0
    assert e.value.code == -2
    ctx = make_ctx()
    with pytest.raises(EfError) as e:                   # expert never registered
        ctx.ef_cache_prefetch(-1, np.ones((1, 8), np.uint8))
    assert e.value.code == -5
    idx = torch.zeros((100, 2), dtype=torch.int32, device="cuda")
    with pytest.raises(EfError) as e:                   # T > max_tokens
        ctx.ef_route_topk(torch.zeros((100, 256), dtype=torch.bfloat16, device="cuda"),
                          torch.zeros((8, 256), dtype=torch.bfloat16, device="cuda"), None, 100, 1, idx,
                          torch.zeros((100, 2), device="cuda"))
    assert e.value.code == -6
    ctx.close()


def test_set_option_validates_keys_and_values():
    from paper_2410_17954_b200 import (EF_OPT_CHUNK_MIN_BYTES, EF_OPT_COPY_ORDER, EF_OPT_FUSED_WAVES, EF_OPT_SPLITK,
                                       EF_OPT_TOKEN_SCHED_PATH, EF_OPT_WAVE_BYTES, EfError)
    ctx = make_ctx()
    for key, good, bad in ((EF_OPT_SPLITK, (0, 1, 16), (-1, 17)), (EF_OPT_WAVE_BYTES, (0, 1 << 40), (-1,)),
                           (EF_OPT_CHUNK_MIN_BYTES, (0, 1), (-5,)), (EF_OPT_COPY_ORDER, (0, 1), (2, -1)),
                           (EF_OPT_FUSED_WAVES, (0, 1), ()), (EF_OPT_TOKEN_SCHED_PATH, (0, 1), ()), (7, (0, 1), ())):   # 7 = EF_OPT_EARLY_RELEASE
        for v in good:
            ctx.ef_set_option(key, v)
        for v in bad:
            with pytest.raises(EfError) as e:
                ctx.ef_set_option(key, v)
            assert e.value.code == -1
    with pytest.raises(EfError):
        ctx.ef_set_option(99, 0)
    ctx.close()


# ------------------------------------------------------------------------------------------------
# diagnostics used by bench.py's second roofline
# ------------------------------------------------------------------------------------------------
def test_tma_fill_rate_and_fill_byte_accounting():
    E, d, f, counts = 2, 512, 1024, [300, 17]
    ctx = make_ctx(n_experts=E, top_k=1, d_model=d, d_ff=f, n_slots=E, max_tokens=int(np.sum(counts)), diag=True)
    gbs = ctx.ef_diag_tma_fill_gbs(32 << 20, 500)
    assert 2000.0 < gbs < 40000.0                     # an L2-resident region: several TB/s on a B200
    with pytest.raises(Exception):
        ctx.ef_diag_tma_fill_gbs(16, 500)             # smaller than one box
    # hand-back between the CTAs of a pair: a cluster-scope RELEASE arrive per stage throttles the stream,
    # a RELAXED one does not -- the reason the grouped GEMM hands ring slots and TMEM halves back with relaxed arrives
    own = ctx.ef_diag_pair_handoff_gbs(32 << 20, 500, 16, -1)
    rel = ctx.ef_diag_pair_handoff_gbs(32 << 20, 500, 16, 0)
    rlx = ctx.ef_diag_pair_handoff_gbs(32 << 20, 500, 16, 1)
    assert rlx > 1.5 * rel and own > rel, (own, rel, rlx)
    with pytest.raises(Exception):
        ctx.ef_diag_pair_handoff_gbs(32 << 20, 500, 15, 1)   # pairs need an even number of CTAs
    ctx.ef_set_kernel_timing(True)
    ctx.ef_get_kernel_times(reset=True)
    run_resident_ffn(ctx, E, d, f, counts, seed=3, simt=False, splitk=1)
    kt = ctx.ef_get_kernel_times(reset=True)
    ctx.ef_set_kernel_timing(False)
    # tile plan (balanced tiles: ceil(rows / 256) tiles of ceil16(rows / tiles) rows): expert 0 = tiles of 160 and 140 rows,
    # expert 1 = one tile of 17 rows.  Per k-block a CTA pair stages 2 x 32 KB of weights (both weight-tile counts are even
    # here: no pair has an idle partner) and, per CTA, the 8 KB token boxes covering half of the tile rounded up to 16 rows
    def per_kb(rows):
        n_mma = (rows + 15) // 16 * 16
        return 2 * (32768 + -(-(n_mma // 2) // 64) * 8192)
    tiles = per_kb(160) + per_kb(140) + per_kb(17)
    npn1, npn2 = (f // 128 + 1) // 2, ((d + 255) // 256 + 1) // 2
    assert kt["gemm1_fill_bytes"] == tiles * npn1 * (d // 64)
    assert kt["gemm2_fill_bytes"] == tiles * npn2 * (f // 64)
    assert kt["wave_rows"] == sum(counts) and kt["wave_groups"] == 2 and kt["wave_launches"] == 1
    assert kt["gemm1_launches"] == 0 and kt["gemm2_launches"] == 0          # one launch ran both GEMMs
    log = ctx.ef_get_launch_log()
    assert [(r["which"], r["groups"], r["rows"]) for r in log] == [(3, 2, sum(counts))] and log[0]["ms"] > 0
    ctx.close()
