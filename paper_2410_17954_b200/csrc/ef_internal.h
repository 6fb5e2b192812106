// Internal declarations shared by libef's translation units.  Not part of the C ABI.
#pragma once

#include <cuda_runtime.h>
#include <cuda.h>
#include <stdint.h>

#include <map>
#include <string>
#include <vector>

#include "ef.h"

#define EF_MAX_GROUPS 64   // groups per grouped-GEMM launch (table travels in kernel params)
#define EF_SCHED_WORDS (1 << 20)  // int32 words of per-launch scheduler blocks {tickets, finished CTAs, one "h rows ready"
                                 // counter per token tile}; self-resetting, carved out of a ring (ffn_tc.cu)
#define EF_W13_BLOCK 128   // gate/up interleave granularity in the packed expert layout

// ---- packed expert layout (library-defined; the caller never sees it) ----------------------------
// An expert occupies W = 3*d*f*2 bytes: the first-GEMM matrix, then the down projection.
//   W13 : 2f rows x d      row 256*j + i       = Wg[128*j + i, :]   (i < 128)
//                          row 256*j + 128 + i = Wu[128*j + i, :]
//         (non-gated experts: W1, f rows x d, rows as given)
//   Wd  : d rows x f       rows as given
// so one 256-row weight tile of GEMM1 yields 128 gate columns and the matching 128 up columns.
// Each matrix M[rows, K] is stored TILED, in the order the grouped GEMM streams it: 256-row tiles, and inside a
// tile one block per 64-column k-block, a block being h x 64 elements row-major (h = 256, or what is left in the
// last tile).  A k-block of a weight tile is therefore 32 KB of CONTIGUOUS memory = one TMA box of 256 "rowlets"
// (a rowlet = 64 bf16 = 128 bytes), instead of 256 rows 2*K bytes apart.  No padding: rows * K elements in all.
#define EF_TILE_ROWS 256
#define EF_ROWLET 64
// element index of M[r, c] inside the tiled matrix
__host__ __device__ inline int64_t ef_tiled_index(int64_t r, int64_t c, int64_t rows, int64_t K) {
    const int64_t t = r / EF_TILE_ROWS, rr = r % EF_TILE_ROWS, kb = c / EF_ROWLET, cc = c % EF_ROWLET;
    const int64_t h = (rows - t * EF_TILE_ROWS < EF_TILE_ROWS) ? rows - t * EF_TILE_ROWS : EF_TILE_ROWS;
    return t * EF_TILE_ROWS * K + kb * h * EF_ROWLET + rr * EF_ROWLET + cc;
}

// One wave of the grouped FFN: group i applies the expert in arena slot `slot` to `rows` token rows that start at
// x_row0 in the input, h_row0 in the h workspace and y_row0 in the output.
struct EfWaveGroup {
    int32_t x_row0, h_row0, y_row0;
    int32_t rows;     // M of this group (> 0)
    int32_t slot;     // arena slot holding the expert
};

struct EfWaveTable {
    int32_t n;
    EfWaveGroup g[EF_MAX_GROUPS];
};

// One slot's policy state (mirror of DESIGN.md §4; written independently of oracle/cache_sim.py).
struct EfSlot {
    int32_t expert = -1;      // global id layer*E + e, or -1
    int64_t pred_for = -1;    // visit the expert was prefetched for; -1: loaded on demand
    bool used = false;        // used since load
    uint64_t stamp = 0;       // tick of last use / of the load
};

// Physical ordering of a slot.  Events come from a ring; a handle whose generation moved on has been
// recycled, and waiting on it falls back to "everything enqueued on the origin stream so far".
struct EvHandle {
    int32_t idx = -1;
    uint32_t gen = 0;
};
struct EfPhys {
    EvHandle ready1;                 // chunked load only: recorded on the copy stream once the first-GEMM weights
                                     // (W13 / W1) have landed, before the copy of Wd starts
    EvHandle ready;                  // recorded on the copy stream after the whole H2D into the slot
    EvHandle free_;                  // recorded on the compute stream after the last wave reading the slot
    bool has_flag = false;           // the slot is handed back from inside its last wave: a copy into it waits for
    uint32_t flag_target = 0;        // *ctx->early_flag to reach this value instead of for `free_`
    uint8_t waited_mask = 0;         // bit 0 / bit 1: stream `waited` has waited on ready1 / ready since the load
    cudaStream_t waited = nullptr;   // (the legacy default stream is a valid value: 0)
};

struct ef_ctx {
    ef_config cfg{};
    int64_t W = 0;                 // bytes per expert
    int32_t n_sms = 148;
    char* arena = nullptr;         // (S + L*n_shared) slots
    int32_t n_arena_slots = 0;
    void* h_ws = nullptr;          // bf16 [h_rows, f]
    int64_t h_rows = 0;
    int32_t* counts_pinned = nullptr;   // pinned mirror of counts[E] + one word of permute error flags
    const int32_t* counts_mirror = nullptr;   // where the last ef_permute mirrored counts (ours or the caller's)
    cudaEvent_t counts_event = nullptr;
    int32_t* permute_ws = nullptr;      // device scratch for ef_permute
    cudaStream_t copy_stream = nullptr;
    std::vector<cudaEvent_t> ev_ring;
    std::vector<uint32_t> ev_gen;
    int32_t ev_next = 0;
    std::vector<EfPhys> phys;           // [S]
    cudaStream_t last_compute = nullptr;   // stream of the layer path's last call (route .. combine); see ef_enter_stream
    bool has_last_compute = false;
    cudaStream_t last_sched = nullptr;     // stream of the token-scheduler path's last call
    bool has_last_sched = false;
    // host pool
    std::vector<void*> host_expert;     // [L*E] packed pinned buffers (owned unless aliased)
    std::vector<char> host_owned;
    std::vector<int32_t> host_aliases;  // [L*E] how many other experts alias this one's buffer
    std::vector<int32_t> alias_src;     // [L*E] the owner an aliasing expert points at, else -1
    std::vector<char> shared_registered;  // [L*n_shared]
    // policy
    std::vector<EfSlot> slots;
    std::vector<int32_t> slot_of;       // [L*E] -> slot or -1
    std::map<int64_t, std::vector<uint8_t>> pred;   // visit -> predicted active flags [E]
    uint64_t tick = 0;
    int32_t policy = EF_POLICY_PLEC;    // ef_set_cache_policy
    ef_cache_stats stats{};
    // tensor map over the whole arena as rowlets (2-D: 64 elements x total rowlets); both GEMMs use it
    CUtensorMap tm_w{};
    CUtensorMap tm_h{};                 // the h workspace [h_rows, f] (fixed for the ctx's life)
    CUtensorMap tm_x{};                 // the caller's x_perm [rows, d], re-encoded only when pointer or row count change
    const void* tm_x_ptr = nullptr;
    int64_t tm_x_rows = 0;
    bool tm_ok = false;
    int32_t* sched_words = nullptr;     // device, [EF_SCHED_WORDS]
    int32_t sched_next = 0;
    // tail split-K of the grouped GEMM (ffn_tc.cu): fp32 partial slots + per-tile arrival counters
    float* splitk_ws = nullptr;
    int32_t* splitk_counters = nullptr;
    int32_t splitk_max_units = 0;
    long long* kprof1 = nullptr;        // -DEF_KPROF builds: per-CTA MMA-warp wait cycles of the last GEMM1 / GEMM2 launch
    long long* kprof2 = nullptr;
    int32_t splitk_mode = 0;            // 0 auto, 1 off, >= 2 force that many K parts on every tile (tests)
    // copy timing
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> copy_spans;
    float copy_ms = 0.f;
    // optional per-launch timing (ef_set_kernel_timing): one pooled event pair per grouped-FFN launch
    int32_t time_kernels = 0;
    struct KSpan { cudaEvent_t e0, e1; int which; int64_t rows; int32_t groups; };   // which: 1 GEMM1, 2 GEMM2, 3 both (one launch)
    std::vector<KSpan> kspans;
    std::vector<cudaEvent_t> timing_pool;    // timing-enabled events, recycled by drain_kernel_spans / drain_copy_spans
    std::vector<ef_launch_record> launch_log;
    ef_kernel_times ktimes{};
    int32_t fused_waves = 1;            // EF_OPT_FUSED_WAVES: 0 = always two launches per wave (test hook)
    // token scheduler workspace (token_sched.cu): state words, packed paths + membership bits, distance matrix
    void* ts_state = nullptr;
    void* ts_small = nullptr;
    size_t ts_small_bytes = 0;
    void* ts_dist = nullptr;
    size_t ts_dist_bytes = 0;
    bool ts_small_attr = false;         // ts_small_kernel opted in to > 48 KB dynamic smem
    void* ts_static_scratch = nullptr;  // device address of token_sched.cu's static scratch array (cudaGetSymbolAddress at ef_create)
    int32_t ts_static_err = 0;          // the cudaError_t of that call
    int32_t ts_force_multi = 0;         // test hook (EF_OPT_TOKEN_SCHED_PATH): 1 = never take the single-CTA path
    // physical scheduling knobs (never part of the policy): ef_set_option(EF_OPT_WAVE_BYTES / EF_OPT_CHUNK_MIN_BYTES)
    int64_t wave_bytes = (int64_t)128 << 20;
    int64_t chunk_min_bytes = (int64_t)32 << 20;
    int32_t copy_order = 1;             // EF_OPT_COPY_ORDER
    int32_t early_release = 1;          // EF_OPT_EARLY_RELEASE
    uint32_t* early_flag = nullptr;     // device word the wave kernel adds finished k-blocks of an early-released slot to
    uint32_t early_target = 0;          // the sum expected so far (host side; compared cyclically)
    void* wait_value_fn = nullptr;      // cuStreamWaitValue32, if the driver has it
    // misc
    int64_t launches = 0;
    int32_t debug_simt = 0;             // diag builds only (ef_diag.h)
    bool route_smem_set = false;        // route kernel opted in to > 48 KB dynamic smem (E > 176)
    std::string err;
    int32_t sticky = EF_OK;
};

int32_t ef_fail(ef_ctx* ctx, int32_t code, const char* fmt, ...);

#define EF_CUDA(ctx, call)                                                                              \
    do {                                                                                                \
        cudaError_t e__ = (call);                                                                       \
        if (e__ != cudaSuccess) {                                                                       \
            (ctx)->sticky = EF_ERR_CUDA;                                                                \
            return ef_fail((ctx), EF_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), \
                           __FILE__, __LINE__);                                                         \
        }                                                                                               \
    } while (0)

#define EF_CHECK_CTX(ctx)                         \
    do {                                          \
        if (!(ctx)) return EF_ERR_INVALID_ARG;    \
        if ((ctx)->sticky != EF_OK) return (ctx)->sticky; \
    } while (0)

// ---- kernels (one launcher per translation unit) ---------------------------------------------------
int32_t efk_route_topk(ef_ctx* ctx, cudaStream_t st, const void* x, const void* wr, const float* bias,
                       int64_t bias_stride, int T, int renorm, int32_t* idx, float* w, float* logits);
int32_t efk_permute(ef_ctx* ctx, cudaStream_t st, const int32_t* idx, const void* x, int T, void* x_perm,
                    int32_t* counts, int32_t* offsets, int32_t* src, int32_t* inv, int32_t* counts_host, int32_t* err_host);
int32_t efk_combine(ef_ctx* ctx, cudaStream_t st, const void* y_perm, const int32_t* inv, const float* w, int T,
                    const void* residual, const void* y_shared, void* out);
int32_t efk_rmsnorm(ef_ctx* ctx, cudaStream_t st, const void* x, int T, float eps, void* out);

// Grouped FFN over arena slots: x rows -> h workspace -> y rows, one wave.
// phase: bit 0 = GEMM1 (x -> h), bit 1 = GEMM2 (h -> y); 3 = both in ONE launch (ffn_tc.cu).
struct EfEarly;
int32_t efk_ffn_grouped(ef_ctx* ctx, cudaStream_t st, const void* x, void* y, const EfWaveTable& tab, int phase, EfEarly* early = nullptr);
#ifdef EF_DIAG
int32_t efk_ffn_simt(ef_ctx* ctx, cudaStream_t st, const void* x, void* y, const EfWaveTable& tab, int phase);
#endif
int32_t efk_timing_events(ef_ctx* ctx, cudaEvent_t* e0, cudaEvent_t* e1);   // a pooled pair of timing-enabled events
int32_t efk_token_schedule(ef_ctx* ctx, cudaStream_t st, const uint8_t* paths, int N, int LE, int c0, int c1,
                           int max_iter, int32_t* batch_of, int32_t* perm, int32_t* info, uint8_t* batch_paths);
int32_t efk_reindex_rows(ef_ctx* ctx, cudaStream_t st, const void* src, const int32_t* perm, int n_rows, int64_t row_bytes,
                         void* dst);
int32_t efk_path_hamming(ef_ctx* ctx, cudaStream_t st, const uint8_t* paths, int N, int LE, uint16_t* dist_out);
void efk_token_sched_free(ef_ctx* ctx);
void efk_token_sched_static_init(ef_ctx* ctx);   // resolves the static scratch's device address; the ctx's device is current
int32_t efk_path_hamming_static(ef_ctx* ctx, cudaStream_t st, const uint8_t* paths, int N, int LE, uint16_t* dist_out);
int32_t efk_ffn_tc_init(ef_ctx* ctx);   // build arena tensor maps, set smem attributes
// Early hand-back of the slot of group 0 from INSIDE a fused wave (ffn_tc.cu, EarlyArgs): the launch adds `add` to
// ctx->early_flag in total, the last of it as soon as nothing of the launch reads that slot any more.
struct EfEarly {
    bool want = false;     // in: hand group 0's slot back early if this wave can
    bool dry = false;      // in: only say whether it could (no launch)
    bool used = false;     // out
    uint32_t add = 0;      // out
};
int32_t efk_ffn_tc(ef_ctx* ctx, cudaStream_t st, const void* x, void* y, const EfWaveTable& tab, int phase, EfEarly* early = nullptr);
