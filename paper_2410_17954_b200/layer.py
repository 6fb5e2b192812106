"""MoELayerRunner: the call a user makes -- one MoE layer visit through libef, in the order of
SURVEY.md §3(ii): route -> permute -> (cache lookup + correction + grouped FFN) -> PLEC prefetch ->
combine.  Sequencing and buffer ownership only; every step of the path runs in the CUDA library.
"""
from __future__ import annotations

import numpy as np
import torch

from .binding import EfContext


def bf16_tensor_from_bits(bits: np.ndarray, device=None, pin=False) -> torch.Tensor:
    """uint16 bit patterns -> torch.bfloat16 tensor (no value conversion)."""
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16)
    if pin:
        t = t.pin_memory()
    if device is not None:
        t = t.to(device, non_blocking=pin)
    return t


def bits_from_bf16_tensor(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


class MoELayerRunner:
    def __init__(self, n_layers, n_experts, top_k, d_model, d_ff, n_slots, n_shared=0, max_tokens=1,
                 prefetch_horizon=0, renorm=1, device=0, expert_kind=0, diag=False):
        if not torch.cuda.is_available():
            raise RuntimeError("MoELayerRunner needs a CUDA device; there is no CPU fallback")
        self.dev = torch.device("cuda", device)
        torch.cuda.set_device(self.dev)
        self.L, self.E, self.k, self.d, self.f = n_layers, n_experts, top_k, d_model, d_ff
        self.n_shared, self.renorm, self.max_tokens = n_shared, renorm, max_tokens
        self.ctx = EfContext(n_layers, n_experts, top_k, d_model, d_ff, n_slots, n_shared, max_tokens,
                             prefetch_horizon, device, expert_kind, diag=diag)
        T, k, E, d = max_tokens, top_k, n_experts, d_model
        dev = self.dev
        self.w_router = [None] * n_layers
        self.bias = [None] * n_layers
        self.topk_idx = torch.empty((T, k), dtype=torch.int32, device=dev)
        self.topk_w = torch.empty((T, k), dtype=torch.float32, device=dev)
        self.logits = torch.empty((T, E), dtype=torch.float32, device=dev)
        self.counts = torch.empty((E,), dtype=torch.int32, device=dev)
        self.offsets = torch.empty((E + 1,), dtype=torch.int32, device=dev)
        self.src = torch.empty((T * k,), dtype=torch.int32, device=dev)
        self.inv = torch.empty((T * k,), dtype=torch.int32, device=dev)
        self.x_perm = torch.empty((T * k, d), dtype=torch.bfloat16, device=dev)
        self.y_perm = torch.empty((T * k, d), dtype=torch.bfloat16, device=dev)
        self.y_shared = torch.empty((max(1, n_shared) * T, d), dtype=torch.bfloat16, device=dev) if n_shared else None
        self.normed = torch.empty((T, d), dtype=torch.bfloat16, device=dev)

    # ---- setup
    def set_router(self, layer, w_router_bits: np.ndarray, bias: np.ndarray | None = None):
        self.w_router[layer] = bf16_tensor_from_bits(w_router_bits, self.dev)
        self.bias[layer] = None if bias is None else torch.from_numpy(np.ascontiguousarray(bias, np.float32)).to(self.dev)

    def register_expert(self, layer, expert, wg, wu, wd):
        self.ctx.ef_host_expert_register(layer, expert, wg, wu, wd)

    # ---- one visit
    def visit(self, visit: int, x: torch.Tensor, out: torch.Tensor, token_bias: torch.Tensor | None = None,
              predicted_next: np.ndarray | None = None, residual: torch.Tensor | None = None,
              want_logits: bool = False, pre_norm_eps: float | None = None):
        """x: [T, d] bf16 device.  out: [T, d] bf16 device.  predicted_next: uint8 [n_ahead, E] for visits
        visit+1.. (None = no prefetch call).  pre_norm_eps: apply RMSNorm to x first (cfg 5 stack)."""
        c = self.ctx
        T = x.shape[0]
        layer = visit % self.L
        inp = x
        if pre_norm_eps is not None:
            inp = self.normed[:T]
            c.ef_rmsnorm(x, T, pre_norm_eps, inp)
        bias = token_bias if token_bias is not None else self.bias[layer]
        c.ef_route_topk(inp, self.w_router[layer], bias, T, self.renorm, self.topk_idx, self.topk_w,
                        self.logits if want_logits else None)
        c.ef_permute(self.topk_idx, inp, T, self.x_perm, self.counts, self.offsets, self.src, self.inv)
        if self.n_shared:
            c.ef_shared_ffn(layer, inp, T, self.y_shared)
        c.ef_expert_ffn_grouped(visit, layer, self.x_perm, None, self.y_perm)
        if predicted_next is not None:
            c.ef_cache_prefetch(visit, predicted_next)
        c.ef_combine(self.y_perm, self.inv, self.topk_w, T, residual, self.y_shared, out)
        return out

    def close(self):
        self.ctx.close()


class DualBatchRunner:
    """Two incoming batches of T tokens per step through the Token Scheduler (§3.3, §4.2): schedule on the
    predicted routing paths -> Reindex activations and per-token rows into the new batches -> the new batches'
    batch-level predicted paths drive the cache prefetch -> 2 x L layer visits.  Sequencing and buffers only.

    Dual-batch pipeline (§4.2, Fig. 6): the scheduling of unit n+1 is interleaved with the decoding of
    unit n -- `schedule_async` enqueues it on a side stream into the other half of double-buffered outputs and
    `wait_schedule` picks the result up when unit n+1 starts, so its cost (kernels, Reindex, the read-back of the
    batch paths) never sits between two decode steps.  `schedule` is the sequential form of the same two calls."""

    def __init__(self, runner: MoELayerRunner, max_iter: int = 8):
        self.r = r = runner
        T, L, E, d, dev = r.max_tokens, r.L, r.E, r.d, r.dev
        self.T, self.N, self.max_iter = T, 2 * T, max_iter
        N = self.N
        self.side = torch.cuda.Stream(device=dev)
        self.batch_of = torch.empty((N,), dtype=torch.int32, device=dev)
        self.perm = torch.empty((N,), dtype=torch.int32, device=dev)
        self.info = torch.empty((8,), dtype=torch.int32, device=dev)
        self.batch_paths = torch.empty((2, L * E), dtype=torch.uint8, device=dev)
        # double-buffered results of a schedule call (slot = unit parity)
        self.batch_paths_host = [torch.empty((2, L * E), dtype=torch.uint8).pin_memory() for _ in range(2)]
        self.x_re_buf = [torch.empty((N, d), dtype=torch.bfloat16, device=dev) for _ in range(2)]
        self.bias_re_buf = [torch.empty((N, L, E), dtype=torch.float32, device=dev) for _ in range(2)]
        self.done = [torch.cuda.Event() for _ in range(2)]
        self.x_re, self.bias_re = self.x_re_buf[0], self.bias_re_buf[0]
        self.hbuf = [torch.empty((T, d), dtype=torch.bfloat16, device=dev) for _ in range(2)]

    def schedule_async(self, pred_paths: torch.Tensor, c0: int, c1: int, x: torch.Tensor, token_bias: torch.Tensor | None,
                       slot: int = 0):
        """Enqueue Token Scheduler + Reindex + batch-path read-back for one dual-batch unit on the side stream, into
        buffer `slot`.  The side stream first waits for everything enqueued on the current stream so far (the inputs'
        producers, and the decode step that last read this slot's buffers).  Returns at once."""
        c = self.r.ctx
        self.side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(self.side):
            c.ef_token_schedule(pred_paths, c0, c1, self.max_iter, self.batch_of, self.perm, self.info, self.batch_paths)
            c.ef_reindex_rows(x, self.perm, self.x_re_buf[slot])
            if token_bias is not None:
                c.ef_reindex_rows(token_bias, self.perm, self.bias_re_buf[slot])
            self.batch_paths_host[slot].copy_(self.batch_paths, non_blocking=True)
            self.done[slot].record(self.side)

    def wait_schedule(self, slot: int = 0):
        """Pick up the result of schedule_async(slot): the current stream waits for the reindexed rows, the host for
        the 2*L*E bytes of batch paths that the (host-side) prefetch call consumes.  Returns the predicted batch-level
        rows uint8 [2L, E] (host) of the unit's 2L visits; x / bias in new-batch order are self.x_re / self.bias_re."""
        torch.cuda.current_stream().wait_event(self.done[slot])
        self.done[slot].synchronize()
        self.x_re, self.bias_re = self.x_re_buf[slot], self.bias_re_buf[slot]
        return self.batch_paths_host[slot].numpy().reshape(2 * self.r.L, self.r.E)

    def schedule(self, pred_paths: torch.Tensor, c0: int, c1: int, x: torch.Tensor, token_bias: torch.Tensor | None):
        """pred_paths uint8 [N, L, E], x bf16 [N, d], token_bias fp32 [N, L, E] (all device).  Sequential form:
        schedule now, wait for it.  Returns what wait_schedule returns."""
        self.schedule_async(pred_paths, c0, c1, x, token_bias, 0)
        return self.wait_schedule(0)

    def run_step(self, step: int, rows: np.ndarray, x: torch.Tensor, token_bias: torch.Tensor | None, out: torch.Tensor,
                 on_visit=None):
        """x [N, d] / token_bias [N, L, E] in batch order (self.x_re / self.bias_re after schedule(), or the incoming
        order for the unscheduled arm); rows uint8 [2L, E] host.  out [N, d]: row i = final hidden state of x row i."""
        r, L, T = self.r, self.r.L, self.T
        v0 = step * 2 * L
        r.ctx.ef_cache_prefetch(v0 - 1, rows)
        for b in range(2):
            h = x[b * T:(b + 1) * T]
            for l in range(L):
                v = v0 + b * L + l
                dst = out[b * T:(b + 1) * T] if l == L - 1 else self.hbuf[l & 1]
                nxt = rows[b * L + l + 1:]
                r.visit(v, h, dst, token_bias=None if token_bias is None else token_bias[b * T:(b + 1) * T, l],
                        predicted_next=nxt if len(nxt) else None, residual=h if L > 1 else None,
                        pre_norm_eps=1e-5 if L > 1 else None)
                if on_visit is not None:
                    on_visit(v, b, l, dst)
                h = dst
        return out
