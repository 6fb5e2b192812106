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
 *   - One ctx per GPU; calls on one ctx must not run concurrently (no two host threads inside the library at once).
 *   - Streams: the library's workspaces are per ctx, not per stream.  The LAYER calls (ef_rmsnorm, ef_route_topk,
 *     ef_permute, ef_expert_ffn_grouped[_resident], ef_shared_ffn, ef_combine) form one lane and the TOKEN-SCHEDULER
 *     calls (ef_token_schedule, ef_path_hamming, ef_reindex_rows) another; the two lanes share nothing and may run
 *     on different streams concurrently.  Inside a lane, a call on a stream other than the lane's previous one is
 *     ordered behind everything the lane has enqueued so far (the library inserts the event wait), so changing
 *     streams is safe but never concurrent.
 *   - CUDA graphs: the memory-bound calls (ef_rmsnorm, ef_route_topk, ef_permute, ef_combine, ef_reindex_rows) may be
 *     issued on a stream that is being captured; the library then inserts no cross-stream ordering (ordering the replayed
 *     graph against other work on the same ctx is the caller's job) and a captured ef_permute leaves no counts mirror
 *     behind for ef_expert_ffn_grouped(counts_host = NULL).  The grouped-FFN calls wait on copy-stream events, and
 *     ef_expert_ffn_grouped on the gate's counts on the host: they are not capturable.
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
 * All device.  counts_host_pinned: nullable PINNED host int32[E] that also receives counts (it must stay valid until
 * the next ef_permute); when NULL the library mirrors counts into its own pinned buffer.  Either way an internal
 * event marks the mirror complete, and ef_expert_ffn_grouped(counts_host = NULL) waits on it and reads that mirror.
 * A topk_idx entry outside [0, E) is not routed anywhere: the pair is skipped (inv = -1) and the next
 * ef_expert_ffn_grouped(counts_host = NULL) fails with EF_ERR_INVALID_ARG. */
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
/* The Hamming distance matrix of Eq. 6 alone: dist_out DEVICE uint16[N, N] (16-byte aligned), d_ij = number of
 * (layer, expert) entries in which r_i and r_j differ; S_ij = 1 - d_ij / LE.  N need not be even here. */
int32_t ef_path_hamming(ef_ctx* ctx, void* stream, const uint8_t* paths, int32_t N, int32_t LE, uint16_t* dist_out);
/* ef_path_hamming for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same result, but the scratch -- the bit-packed paths, N * ceil(LE / 32) * 4 bytes --
 * lives in a static device array inside the library instead of in a cudaMalloc'ed workspace.  The call makes no
 * cudaMalloc, cudaFree or allocating library call: it launches two kernels on `stream`.
 *   - Limit: N * ceil(LE / 32) * 4 <= EF_STATIC_SCRATCH_BYTES (1 MiB; e.g. N = 4096 tokens of LE = 2048 path entries);
 *     beyond it the call fails with EF_ERR_CAPACITY and does nothing.  The array costs that much memory on every GPU that
 *     loads the library, until the process exits.
 *   - Its device address is resolved once per ctx at ef_create (cudaGetSymbolAddress with the ctx's device current); if
 *     that failed, this call returns EF_ERR_CUDA with the reason.
 *   - ONE array per device, shared by every call and every ctx on that device: two calls that overlap on the GPU (two
 *     streams, two ctxs, two host threads) race on it and both results are undefined; calls on one stream are safe.  The
 *     array keeps the last call's contents; nothing in it has to start at zero (every word read is written first). */
#define EF_STATIC_SCRATCH_BYTES (1 << 20)
int32_t ef_path_hamming_static(ef_ctx* ctx, void* stream, const uint8_t* paths, int32_t N, int32_t LE, uint16_t* dist_out);

/* ---- misc ---------------------------------------------------------------------------------- */
/* Wait for the copy stream and the device.  Synchronous. */
int32_t ef_sync(ef_ctx* ctx);
/* Text of the last error on ctx (ctx may be NULL: last ef_create failure).  Never NULL. */
const char* ef_last_error(ef_ctx* ctx);
/* Number of kernels this ctx has launched since creation (for bench.py's gpu_launches). */
int64_t ef_launch_count(ef_ctx* ctx);
/* Per-launch device timing of the grouped FFN, for roofline reporting (bench.py).  When on, every grouped-FFN launch is
 * bracketed by CUDA events on the compute stream.  A wave is ONE launch that runs both GEMMs (`which` = 3); a wave whose
 * expert is still arriving in two chunks runs GEMM1 (`which` = 1) and GEMM2 (`which` = 2) as two launches gated on
 * different events.  ef_get_kernel_times waits for the recorded events (synchronous), returns the totals since the last
 * reset and optionally resets; ef_get_launch_log returns the same launches one by one (oldest first), so that a caller can
 * hold every launch against ITS OWN roofline bound max(FLOP / peak, bytes / bandwidth).
 * Algorithmic work of a launch over `rows` routed rows in `groups` experts (SwiGLU): GEMM1 4*d*f FLOP per row and 4*d*f
 * weight bytes per group, GEMM2 2*d*f and 2*d*f (ReLU experts: 2*d*f for both GEMMs). */
typedef struct {
    double gemm1_ms, gemm2_ms, wave_ms;               /* device time of the which = 1 / 2 / 3 launches */
    int64_t gemm1_launches, gemm2_launches, wave_launches;
    int64_t gemm1_rows, gemm2_rows, wave_rows;        /* routed rows those launches processed */
    int64_t gemm1_groups, gemm2_groups, wave_groups;  /* expert groups those launches processed */
    int64_t gemm1_fill_bytes, gemm2_fill_bytes;       /* bytes the launches' TMA loads staged into shared memory for GEMM1 /
                         GEMM2 units (weight boxes + token boxes over every tile and k-block, from the tile plan): the
                         L2 -> SM traffic */
} ef_kernel_times;
typedef struct {
    int32_t which;     /* 1 GEMM1 only, 2 GEMM2 only, 3 both GEMMs in one launch */
    int32_t groups;    /* experts in the launch */
    int64_t rows;      /* routed rows in the launch */
    float ms;          /* device time between the events around the launch */
} ef_launch_record;
int32_t ef_set_kernel_timing(ef_ctx* ctx, int32_t on);
int32_t ef_get_kernel_times(ef_ctx* ctx, ef_kernel_times* out, int32_t reset);
/* out: HOST ef_launch_record[max_records]; *n_out = records written (the log keeps at most 65536).  Synchronous. */
int32_t ef_get_launch_log(ef_ctx* ctx, ef_launch_record* out, int32_t max_records, int32_t* n_out, int32_t reset);

/* Physical-scheduling knobs and test hooks.  None of them changes what is computed or any cache counter (results differ
 * between EF_OPT_SPLITK settings only by fp32 summation order):
 * EF_OPT_SPLITK          tail split-K of the grouped GEMM: 0 = automatic (default: the tiles of the last,
 *                        partly filled round are split along K so that every SM stays busy), 1 = never, 2..16 = split
 *                        EVERY tile into that many K parts (test hook: exercises the partial-sum workspace on small shapes).
 * EF_OPT_WAVE_BYTES      consecutive on-demand experts of a visit are computed by one grouped launch per `value` bytes of
 *                        expert weights on the link (default 128 MiB; an expert larger than that, and always the last
 *                        miss of a visit, is its own launch; 0 = one launch per miss) -- SURVEY.md 8(f).3.
 * EF_OPT_CHUNK_MIN_BYTES experts of at least `value` bytes (default 32 MiB) are copied as two chunks -- first-GEMM weights,
 *                        then the down projection -- each with its own "ready" event, so GEMM1 of the visit's last wave
 *                        overlaps the second chunk's transfer (0 = always one copy per expert).
 * EF_OPT_FUSED_WAVES     1 (default) = a wave is one launch running both GEMMs; 0 = always two launches (test hook).
 * EF_OPT_TOKEN_SCHED_PATH problems with N <= 256 (decode batches) run in one single-CTA kernel with the distance matrix in
 *                        shared memory, larger ones in the multi-kernel path; 1 = always the multi-kernel path (test hook).
 * EF_OPT_COPY_ORDER      order in which the on-demand copies of one visit are put on the link: 0 = policy order (ascending
 *                        expert id, R12), 1 (default) = experts with more routed rows first, so the largest GEMMs start
 *                        earliest (the paper's "high-priority queue").  Which slot an expert takes
 *                        and every counter are decided in policy order either way.
 * EF_OPT_EARLY_RELEASE   1 (default) = the hit whose slot the visit's first pending copy will overwrite is handed back from
 *                        INSIDE the hits' wave (its units are ticketed first and count themselves done on a device word
 *                        the copy stream waits for) when that hit is a decode-sized expert (one token tile of <= 128 rows);
 *                        0 = that hit always runs as a wave of its own first.
 *                        Physical scheduling only. */
#define EF_OPT_SPLITK 1
#define EF_OPT_WAVE_BYTES 2
#define EF_OPT_CHUNK_MIN_BYTES 3
#define EF_OPT_FUSED_WAVES 4
#define EF_OPT_TOKEN_SCHED_PATH 5
#define EF_OPT_COPY_ORDER 6
#define EF_OPT_EARLY_RELEASE 7
int32_t ef_set_option(ef_ctx* ctx, int32_t key, int64_t value);

#ifdef __cplusplus
}
#endif
#endif /* EF_H_ */
