"""The seeded input generators: determinism, storage-format conversions, and the statistical structure
DESIGN.md §5 promises (skew, temporal locality, predictor accuracy).  CPU only."""
import numpy as np

import workloads as wl


def test_deterministic_and_order_independent():
    cfg = wl.CONFIGS["tiny"]
    a = wl.expert_weights(cfg, 0, 3)
    _ = wl.activations(cfg)
    b = wl.expert_weights(cfg, 0, 3)
    for u, v in zip(a, b):
        assert np.array_equal(u, v)
    assert not np.array_equal(a[0], wl.expert_weights(cfg, 0, 4)[0])
    assert not np.array_equal(wl.activations(cfg, 0), wl.activations(cfg, 1))


def test_bf16_roundtrip_and_rne():
    v = np.array([1.0, -2.5, 0.0, 3.140625], np.float32)    # all exactly representable in bf16
    assert np.array_equal(wl.bf16_bits_to_f32(wl.f32_to_bf16_bits(v)), v)
    x = wl.stream(1, "x").standard_normal(100000).astype(np.float32)
    back = wl.bf16_bits_to_f32(wl.f32_to_bf16_bits(x))
    assert np.all(np.abs(back - x) <= np.abs(x) * 2.0 ** -8)   # half ulp of an 8-bit significand


def test_distributions():
    cfg = wl.CONFIGS["tiny"]
    wg, _, _ = wl.expert_weights(cfg, 0, 0)
    assert abs(wl.bf16_bits_to_f32(wg).std() - 0.02) < 1e-3
    wr = wl.bf16_bits_to_f32(wl.router_weight(cfg))
    assert abs(wr.std() - 1 / 16) < 5e-3
    z = wl.static_router_bias(wl.CONFIGS["many_expert_prefill"])
    assert z.shape == (64,) and np.isclose(np.sort(z)[::-1][1], -1.1 * np.log(2), atol=1e-6)
    assert wl.static_router_bias(cfg) is None


def test_trace_structure():
    cfg = wl.scaled(wl.CONFIGS["mixtral_decode"], d_model=64, d_ff=128)
    tr = wl.routing_trace(cfg, 200)
    assert tr.sets.shape == (200, 16, 2)
    assert all(len(set(s)) == 2 for s in tr.sets.reshape(-1, 2).tolist())   # distinct experts per token
    same = np.mean([set(a) == set(b) for a, b in zip(tr.sets[1:].reshape(-1, 2).tolist(),
                                                      tr.sets[:-1].reshape(-1, 2).tolist())])
    assert 0.55 < same < 0.80                       # keep_prob 0.6 plus chance re-draws
    b = wl.trace_bias(cfg, tr, 5)
    top2 = np.argsort(-b, axis=1)[:, :2]
    assert np.array_equal(top2, tr.sets[5])
    # batch-level recall of the predicted path (PAPER Eq. 7 style) sits between token accuracy and 1
    rec = (tr.predicted & tr.actual).sum() / tr.actual.sum()
    assert 0.85 <= rec <= 1.0
