/*
 * ef.h -- C ABI of libef: the MoE expert layer running against a GPU-resident expert cache
 * (ExpertFlow, arxiv 2410.17954), hand-written CUDA for sm_100a (B200).
 *
 * Citations: P:L<n> = PAPER.md line n.  R<n> = reading n in DESIGN.md §3 (where the paper is silent).
 *
 * Conventions
 *   - Every function returns int32_t: EF_OK (0) or a negative EF_ERR_* code.  No exceptions, no
 *     aborts, no output on stdout.  ef_last_error(ctx) returns text for the last failure.
 *   - "device" pointers are CUDA device pointers on ctx's device, 16-byte aligned, row-major,
 *     contiguous.  "host" pointers are ordinary host memory unless "pinned" is stated.
 *   - bf16 tensors are passed as `const void*` / `void*` (2 bytes per element).
 *   - `stream` is a cudaStream_t passed as void* (e.g. torch.cuda.current_stream().cuda_stream).
 *     All device work of a call is enqueued on it and the call returns without waiting, unless
 *     "synchronous" is stated.  Weight copies run on the library's own copy stream and are ordered
 *     against `stream` with events.
 *   - Ownership: the caller owns every activation / index buffer.  The library owns the slot
 *     arena, copy stream, events, workspaces, the slot table and -- after ef_host_expert_register --
 *     a packed copy of each expert in its own pinned host pool (every expert is backed up
 *     on the host, so eviction needs no write-back).
 *   - One ctx per GPU; calls on one ctx must not run concurrently.
 *   - Shape limits: d_model % 64 == 0, d_ff % 128 == 0, 1 <= top_k <= 8, top_k <= n_experts <= 256.
 *
 * Logical clock: visit = step * n_layers + layer.  The cache policy depends only on the sequence
 * of calls and their arguments, never on whether a copy or kernel has physically finished (R9).
 */
#ifndef EF_H_
#define EF_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EF_OK 0
#define EF_ERR_INVALID_ARG (-1)
#define EF_ERR_UNSUPPORTED (-2)    /* shape / alignment outside the limits above */
#define EF_ERR_CUDA (-3)           /* a CUDA call failed; sticky */
#define EF_ERR_OOM (-4)
#define EF_ERR_NOT_REGISTERED (-5) /* an expert that must be loaded was never registered */
#define EF_ERR_CAPACITY (-6)       /* more tokens than max_tokens, more groups than slots, ... */

typedef struct ef_ctx ef_ctx;

typedef struct {
    int32_t n_layers;          /* L: layers sharing the one global slot pool (R7) */
    int32_t n_experts;         /* E: routed experts per layer */
    int32_t top_k;             /* k */
    int32_t d_model;           /* d */
    int32_t d_ff;              /* f */
    int32_t n_slots;           /* S: cache slots, each holds one routed expert (3*d*f*2 bytes) */
    int32_t n_shared;          /* always-resident shared experts per layer, outside the pool (R19) */
    int32_t max_tokens;        /* largest T of any call */
    int32_t prefetch_horizon;  /* H: visits ahead ef_cache_prefetch may load for; <= 0: as far as supplied (R10) */
    int32_t device;            /* CUDA device ordinal */
    int32_t expert_kind;       /* 0: SwiGLU expert (w_gate, w_up, w_down), 3*d*f*2 bytes (BASELINE.json; R4);
                                  1: Switch-style non-gated ReLU expert y = relu(x W1^T) W2^T (w_gate = W1, w_up = NULL,
                                  w_down = W2), 2*d*f*2 bytes (R30; the paper's Switch-32/64/128 models) */
} ef_config;

typedef struct {
    uint64_t lookups;          /* active (visit, expert) pairs seen by ef_expert_ffn_grouped (R6) */
    uint64_t hits;             /* ... found in the slot table (present or in flight) */
    uint64_t misses;           /* ... not found: loaded on demand ("on-demand experts") */
    uint64_t prefetch_issued;  /* loads started by ef_cache_prefetch */
    uint64_t prefetch_used;    /* prefetched experts whose first use was a hit */
    uint64_t prefetch_wasted;  /* prefetched experts evicted before any use ("mis-prefetched") */
    uint64_t ondemand_loads;   /* == misses */
    uint64_t evictions;        /* occupied slots overwritten or dropped */
    uint64_t bytes_h2d;        /* bytes copied host -> device for expert weights */
} ef_cache_stats;

/* ---- lifetime ------------------------------------------------------------------------------ */

/* Allocates the slot arena ((S + L*n_shared) * 3*d*f*2 bytes), workspaces, copy stream, events.
 * Synchronous.  *out is NULL on failure. */
int32_t ef_create(const ef_config* cfg, ef_ctx** out);
int32_t ef_destroy(ef_ctx* ctx);

/* Register expert `expert` of `layer` (expert < 0: shared expert -1-expert, which is also copied to
 * its resident device slot).  w_gate, w_up: [f, d] bf16; w_down: [d, f] bf16; HOST pointers, read
 * during the call only (the library packs them into its pinned pool).  With expert_kind = 1 (non-gated
 * ReLU expert, R30) w_gate is W1, w_down is W2 and w_up must be NULL.  Synchronous. */
int32_t ef_host_expert_register(ef_ctx* ctx, int32_t layer, int32_t expert, const void* w_gate,
                                const void* w_up, const void* w_down);

/* Make (layer, expert) share the packed host buffer already registered for (src_layer, src_expert):
 * lets a 90 GB logical pool (BASELINE.json cfg 5) run on a host that cannot pin that much.  Bytes
 * moved, policy and accounting are unchanged. */
int32_t ef_host_expert_alias(ef_ctx* ctx, int32_t layer, int32_t expert, int32_t src_layer, int32_t src_expert);

/* ---- a1: router (Eq. 1-2; top-k per P:L52; R1-R3) -------------------------------- */

/* logits[t,e] = sum_c x[t,c] * w_router[e,c] + bias[t*bias_token_stride + e]   (fp32 accumulate)
 * topk_idx[t,:] = the k largest logits' experts, descending, ties -> lower index (R2)
 * topk_w[t,j]   = exp(l_j - max) / Z,  Z over the k selected (renorm=1) or over all E (renorm=0, Eq. 1)
 * x: [T, d] bf16 device.  w_router: [E, d] bf16 device.  bias: fp32 device, nullable;
 * bias_token_stride 0 (per expert, [E]) or >= E floats (per token; E for a dense [T,E], larger to select one layer of a
 * [T,L,E] tensor).  topk_idx: [T,k] int32, topk_w: [T,k]
 * fp32, logits_out: [T,E] fp32 nullable -- all device.  T may be 0. */
int32_t ef_route_topk(ef_ctx* ctx, void* stream, const void* x, const void* w_router, const float* bias,
                      int64_t bias_token_stride, int32_t T, int32_t renorm, int32_t* topk_idx, float* topk_w,
                      float* logits_out);

/* ---- a2: permute (dispatch implied by P:L21; R5) ------------------------------------- */

/* Stable counting sort of the flat pairs p = t*k + j by topk_idx[p]:
 *   counts[E], offsets[E+1] (exclusive scan), inv[p] = row, src[row] = p, x_perm[row,:] = x[p / k,:].
 * All device.  counts_host_pinned: nullable PINNED host int32[E] that also receives counts; when
 * NULL the library mirrors counts into its own pinned buffer.  Either way an internal event marks
 * the mirror complete and ef_expert_ffn_grouped(counts_host = NULL) waits on it. */
int32_t ef_permute(ef_ctx* ctx, void* stream, const int32_t* topk_idx, const void* x, int32_t T, void* x_perm,
                   int32_t* counts, int32_t* offsets, int32_t* src, int32_t* inv, int32_t* counts_host_pinned);

/* ---- a3 + a4: cache lookup, real-time correction, grouped SwiGLU expert FFN ----------------- */

/* For each expert e of `layer` with counts[e] > 0, rows [offsets[e], offsets[e+1]) of x_perm:
 *   y_perm[r,:] = ( silu(x_perm[r,:] Wg_e^T) * (x_perm[r,:] Wu_e^T) ) Wd_e^T      (bf16 in, fp32 accumulate)
 * with the weights read from the cache slot holding (layer, e).  Experts not resident are loaded on
 * demand into victim slots (victim classes R8-R13) on the copy stream while resident
 * experts compute; compute is issued in waves gated by per-slot events.  Updates the counters.
 * counts_host: host int32[E] (what the gate actually selected); NULL = use the mirror written by the
 * last ef_permute, which makes this call wait for that kernel (the one device->host sync per visit,
 * P:L128 "based on the MoE gate's output").  x_perm: [T*k, d] bf16 device; y_perm: [T*k, d] bf16 device.
 * The intermediate h lives in a library workspace. */
int32_t ef_expert_ffn_grouped(ef_ctx* ctx, void* stream, int64_t visit, int32_t layer, const void* x_perm,
                              const int32_t* counts_host, void* y_perm);

/* Kernel-only variant for roofline timing and stage tests: no lookup, no loads, no counters.
 * Group i applies the expert held in cache slot slots[i] to rows [row_begin[i], row_begin[i]+rows[i]).
 * row_begin, rows, slots: HOST int32[n_groups]. */
int32_t ef_expert_ffn_grouped_resident(ef_ctx* ctx, void* stream, const void* x_perm, int32_t n_groups,
                                       const int32_t* row_begin, const int32_t* rows, const int32_t* slots,
                                       void* y_perm);

/* Shared experts of `layer` applied to every token (R19): y_shared[s*T + t, :] = FFN_shared_s(x[t,:]).
 * x: [T,d] bf16 device; y_shared: [n_shared*T, d] bf16 device. */
int32_t ef_shared_ffn(ef_ctx* ctx, void* stream, int32_t layer, const void* x, int32_t T, void* y_shared);

/* ---- a5: combine (Eq. 2 summed over the k selected experts) --------------------------------- */

/* out[t,:] = residual[t,:] + sum_j topk_w[t,j] * y_perm[inv[t*k+j],:] + sum_s y_shared[s*T+t,:]
 * accumulated in fp32, rounded to bf16 once.  residual, y_shared nullable.  All device. */
int32_t ef_combine(ef_ctx* ctx, void* stream, const void* y_perm, const int32_t* inv, const float* topk_w,
                   int32_t T, const void* residual, const void* y_shared, void* out);

/* ---- a8: RMSNorm with unit gain between layers (BASELINE.json cfg 5; R19) ------------------- */
int32_t ef_rmsnorm(ef_ctx* ctx, void* stream, const void* x, int32_t T, float eps, void* out);

/* ---- a6 / a7: cache manager (P:L116-124 PLEC, P:L183-187 overlap, P:L338 no write-back) ------ */

/* PLEC refill after visit `visit_now` (-1 before the first visit).  predicted: HOST uint8[n_ahead, E],
 * row i = batch-level predicted path of visit visit_now+1+i (nonzero = predicted active).  For each
 * visit in order (at most prefetch_horizon of them), each predicted expert (ascending) that is not
 * resident gets a victim slot (empty -> mis-prefetched -> completed with a later next use) and an H2D
 * copy on the copy stream; stops at the first expert with no victim.  Returns immediately. */
int32_t ef_cache_prefetch(ef_ctx* ctx, int64_t visit_now, const uint8_t* predicted, int32_t n_ahead);

/* Drop experts of `layer` from the slot table (no write-back).  experts: HOST int32[n]. */
int32_t ef_cache_evict(ef_ctx* ctx, int32_t layer, const int32_t* experts, int32_t n);

int32_t ef_cache_get_stats(ef_ctx* ctx, ef_cache_stats* out);
int32_t ef_cache_reset_stats(ef_ctx* ctx);
/* slot_to_expert: HOST int32[S]; global expert id layer*E + e, or -1 if empty. */
int32_t ef_cache_snapshot(ef_ctx* ctx, int32_t* slot_to_expert);
/* Empty the slot table and forget supplied predictions (counters untouched). */
int32_t ef_cache_clear(ef_ctx* ctx);

/* Replacement policy of the slot table.  EF_POLICY_PLEC (default) is the paper's Expert Cache Engine as read
 * in DESIGN.md section 4.  The other two are the baselines the paper compares against, as policy sketches on the same
 * machinery: on-demand loading with least-recently-used replacement over the whole
 * pool (EF_POLICY_LRU) or inside a fixed share of n_slots / n_layers slots per layer (EF_POLICY_LAYER_LRU, "fixed-size
 * cache per layer"); under both, ef_cache_prefetch accepts its arguments and does nothing.  (The third baseline of
 * P:L230, prefetching ALL experts of the next layer, needs no policy: it is EF_POLICY_PLEC with an all-ones predicted path
 * and prefetch_horizon = 1.)  Only allowed while the slot table is empty. */
#define EF_POLICY_PLEC 0
#define EF_POLICY_LRU 1
#define EF_POLICY_LAYER_LRU 2
int32_t ef_set_cache_policy(ef_ctx* ctx, int32_t policy);

/* Device time the copy stream spent on expert loads since the last reset, from events (milliseconds),
 * and the wall time of the window in which the copy queue was non-empty are not part of parity;
 * ef_copy_busy_ms waits for the copy stream.  Synchronous. */
int32_t ef_copy_busy_ms(ef_ctx* ctx, float* ms_out);

/* ---- f1: Token Scheduler (Sec. 3.3) ------------------
 * N = 2T tokens (two incoming batches: tokens [0, T) and [T, 2T)), each with a binary routing-path matrix r_i of
 * size (L, E), are split into two new batches of exactly T tokens so that fewer experts are activated
 * (Eq. 5).  Heuristic of Sec. 3.3.3: Hamming distance d_ij between paths, similarity
 * S_ij = 1 - d_ij / (L*E) (Eq. 6); balanced 2-means whose centroids are tokens: assign every token to the more
 * similar centroid, rebalance to exactly T per cluster (R26: cluster 0 = the T tokens with the largest
 * S[i,c0] - S[i,c1]; R27: ties to the lower index), move each centroid to the member with the highest average
 * similarity to the others (R27/R29), stop when the centroids repeat (R28) or after max_iter rounds.
 *
 * paths     DEVICE uint8[N, LE], LE = L*E, row-major, nonzero = expert on the path (the predictor's output)
 * c0, c1    the two distinct tokens drawn as initial centroids ("random centroid selection": the draw is
 *           the caller's, so that results are reproducible)
 * batch_of  DEVICE int32[N]  out: 0 or 1
 * perm      DEVICE int32[N]  out: tokens of new batch 0 in ascending index, then those of new batch 1 -- the
 *           gather map for activations / the KV-cache "Reindex" of P:L151
 * info      DEVICE int32[8]  out: {rounds executed, converged (0/1), final c0, final c1, Eq. 5 objective of the
 *           result, Eq. 5 objective of the incoming batching, 0, 0}; batch-level paths combine tokens with OR (R14)
 * batch_paths DEVICE uint8[2, LE] out, nullable: the batch-level routing paths R_1, R_2 of Eq. 4 (0/1) of the new
 *           batches -- what ef_cache_prefetch wants as the predicted path of each batch's visits
 * Constraints: N even, 2 <= N <= EF_TS_MAX_TOKENS, 1 <= LE <= 32767, 1 <= max_iter <= 64.  Asynchronous on
 * `stream`; the library owns the workspace (bit-packed paths, the uint16 N x N distance matrix). */
#define EF_TS_MAX_TOKENS 16384
int32_t ef_token_schedule(ef_ctx* ctx, void* stream, const uint8_t* paths, int32_t N, int32_t LE, int32_t c0,
                          int32_t c1, int32_t max_iter, int32_t* batch_of, int32_t* perm, int32_t* info,
                          uint8_t* batch_paths);
/* "Reindex": dst row i = src row perm[i] for i < n_rows -- moves activations (and any other per-token rows:
 * router bias, KV entries) into the order of the new batches.  src, dst DEVICE, rows of row_bytes bytes (multiple of
 * 16, 16-byte aligned), out of place; perm DEVICE int32[n_rows] (need not be a permutation).  Asynchronous. */
int32_t ef_reindex_rows(ef_ctx* ctx, void* stream, const void* src, const int32_t* perm, int32_t n_rows,
                        int64_t row_bytes, void* dst);
/* Problems with N <= 256 (decode batches) run in one single-CTA kernel with the distance matrix in shared memory;
 * larger ones in the multi-kernel path.  Test hook: 1 = always take the multi-kernel path.  Results are identical. */
int32_t ef_set_token_sched_path(ef_ctx* ctx, int32_t force_multi_kernel);
/* The Hamming distance matrix of Eq. 6 alone: dist_out DEVICE uint16[N, N] (16-byte aligned), d_ij = number of
 * (layer, expert) entries in which r_i and r_j differ; S_ij = 1 - d_ij / LE.  N need not be even here. */
int32_t ef_path_hamming(ef_ctx* ctx, void* stream, const uint8_t* paths, int32_t N, int32_t LE, uint16_t* dist_out);

/* ---- misc ---------------------------------------------------------------------------------- */
/* Wait for the copy stream and the device.  Synchronous. */
int32_t ef_sync(ef_ctx* ctx);
/* Text of the last error on ctx (ctx may be NULL: last ef_create failure).  Never NULL. */
const char* ef_last_error(ef_ctx* ctx);
/* Number of kernels this ctx has launched since creation (for bench.py's gpu_launches). */
int64_t ef_launch_count(ef_ctx* ctx);
/* Per-kernel device timing of the grouped FFN, for roofline reporting (bench.py).  When on, every
 * grouped-GEMM launch is bracketed by CUDA events on the compute stream.  ef_get_kernel_times waits for
 * the recorded events (synchronous), returns the totals since the last reset and optionally resets.
 * rows = sum over launches of the routed rows they processed (algorithmic FLOPs: gemm1 4*d*f per row,
 * gemm2 2*d*f per row; algorithmic weight bytes: groups * 3*d*f*2). */
typedef struct {
    double gemm1_ms, gemm2_ms;
    int64_t gemm1_launches, gemm2_launches;
    int64_t rows;     /* routed rows processed (each counted once per FFN, not per GEMM) */
    int64_t groups;   /* expert groups processed */
    int64_t gemm1_fill_bytes, gemm2_fill_bytes;   /* bytes the launches' TMA loads staged into shared memory (weight
                         boxes + token boxes over every tile and k-block, from the tile plan): the L2 -> SM traffic */
} ef_kernel_times;
int32_t ef_set_kernel_timing(ef_ctx* ctx, int32_t on);
int32_t ef_get_kernel_times(ef_ctx* ctx, ef_kernel_times* out, int32_t reset);
/* Tail split-K of the grouped GEMM: 0 = automatic (default: split the tiles of the last, partly
 * filled round along K so that every SM stays busy), 1 = never split, 2..16 = split EVERY tile into that many
 * K parts (test hook: exercises the partial-sum workspace on small shapes).  Results differ between modes only
 * by fp32 summation order. */
int32_t ef_set_splitk(ef_ctx* ctx, int32_t mode);
/* Physical scheduling of on-demand loads (never part of the policy or its counters):
 * ef_set_wave_bytes: consecutive on-demand experts of a visit are computed by one grouped launch per `bytes` of
 *   expert weights on the link (default 128 MiB; an expert larger than that, and always the last miss of a visit, is
 *   its own launch; 0 = one launch pair per miss).
 * ef_set_chunk_min_bytes: experts of at least `bytes` (default 32 MiB) are copied as two chunks -- first-GEMM weights,
 *   then the down projection -- each with its own "ready" event, so GEMM1 overlaps the second chunk's transfer
 *   (0 = always one copy per expert).  Results are identical in every setting. */
int32_t ef_set_wave_bytes(ef_ctx* ctx, int64_t bytes);
int32_t ef_set_chunk_min_bytes(ef_ctx* ctx, int64_t bytes);
/* Diagnostic: the rate at which TMA can fill shared memory on this device, i.e. the L2 -> SM fabric ceiling that bounds
 * the grouped GEMM's operand traffic.  One persistent CTA per SM streams 32 KB boxes (64 x 256 bf16, the
 * GEMM's weight box) through a 4-stage ring, `iters` boxes per CTA, out of a scratch region of region_bytes (<= 126 MB
 * stays in L2; larger streams from HBM).  gbs_out: HOST double, delivered GB/s.  Synchronous; allocates and frees the
 * region. */
int32_t ef_debug_tma_fill_gbs(ef_ctx* ctx, int64_t region_bytes, int32_t iters, double* gbs_out);
/* Diagnostic, only in libraries built with -DEF_KPROF (EF_ERR_UNSUPPORTED otherwise): the first call arms the
 * counters, later calls return, per CTA of the last GEMM1 (which = 1) or GEMM2 (which = 2) launch, the cycles the
 * MMA-issuing lane spent {in total, waiting for a tile ticket, waiting for the epilogue to free TMEM, waiting for
 * TMA to fill a stage} and the units it processed.  out: HOST int64[5 * SM count].  Synchronous. */
int32_t ef_debug_kprof(ef_ctx* ctx, int32_t which, int64_t* out);
/* 0 = tcgen05 kernels (default); 1 = plain-FMA debug kernels for the grouped FFN (bring-up aid, slow). */
int32_t ef_set_debug_simt_ffn(ef_ctx* ctx, int32_t on);

#ifdef __cplusplus
}
#endif
#endif /* EF_H_ */
