// libef: context, host expert pool, cache manager (policy + copy-stream pipeline) and the C ABI.
//
// The cache manager implements DESIGN.md §4 (§3.2.1 PLEC, §3.2.2 real-time correction,
// §4.1 multi-stream overlap) on its own; oracle/cache_sim.py is an independent restatement used
// only by the tests.  Every policy decision depends on the call sequence alone (R9): "completed"
// means enqueued, physical ordering is enforced with events:
//   ready event  -- recorded on the copy stream after an expert's H2D; the compute stream waits on it
//   free  event  -- recorded on the compute stream after the last wave reading a slot; the copy
//                   stream waits on it before overwriting the slot.
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <tuple>

#include "ef_internal.h"

static std::string g_create_err;

int32_t ef_fail(ef_ctx* ctx, int32_t code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf; else g_create_err = buf;
    return code;
}

// ---------------------------------------------------------------------------------------------------
// event ring with generations
// ---------------------------------------------------------------------------------------------------
constexpr int kRing = 2048;

static EvHandle ring_record(ef_ctx* ctx, cudaStream_t st, cudaError_t* err) {
    const int i = ctx->ev_next;
    ctx->ev_next = (ctx->ev_next + 1) % kRing;
    ctx->ev_gen[i]++;
    *err = cudaEventRecord(ctx->ev_ring[i], st);
    return EvHandle{i, ctx->ev_gen[i]};
}

// make `waiter` wait for handle h (recorded on `origin`); if h was recycled, wait for everything
// enqueued on `origin` so far, which is a superset.
static cudaError_t ring_wait(ef_ctx* ctx, cudaStream_t waiter, const EvHandle& h, cudaStream_t origin,
                             bool origin_valid = true) {
    if (h.idx < 0) return cudaSuccess;
    if (ctx->ev_gen[h.idx] == h.gen) return cudaStreamWaitEvent(waiter, ctx->ev_ring[h.idx], 0);
    if (!origin_valid || origin == waiter) return cudaSuccess;
    cudaError_t e;
    EvHandle f = ring_record(ctx, origin, &e);
    if (e != cudaSuccess) return e;
    return cudaStreamWaitEvent(waiter, ctx->ev_ring[f.idx], 0);
}

// The library's workspaces are per ctx, not per stream (ef.h, "Streams").  Every stream-taking call of a lane passes
// through here first: a call on a stream other than the lane's previous one is ordered behind everything the lane has
// enqueued so far, so that two streams can never interleave inside the split-K workspace, the h workspace, the
// scheduler blocks or a slot that a copy is about to overwrite.
static int32_t enter_lane(ef_ctx* ctx, cudaStream_t st, cudaStream_t* last, bool* has_last) {
    // A stream that is being captured into a CUDA graph executes nothing now: ordering the replayed graph against the
    // lane's other work is the capturer's business (ef.h), and an event recorded outside the capture could not be waited
    // on from inside it anyway.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap == cudaStreamCaptureStatusActive) return EF_OK;
    if (*has_last && *last != st) {
        cudaError_t e;
        EvHandle h = ring_record(ctx, *last, &e);
        EF_CUDA(ctx, e);
        EF_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_ring[h.idx], 0));
    }
    *last = st;
    *has_last = true;
    return EF_OK;
}
#define EF_ENTER_LAYER(ctx, st)                                                                   \
    do {                                                                                          \
        int32_t rc__ = enter_lane((ctx), (st), &(ctx)->last_compute, &(ctx)->has_last_compute);  \
        if (rc__ != EF_OK) return rc__;                                                           \
    } while (0)
#define EF_ENTER_SCHED(ctx, st)                                                               \
    do {                                                                                      \
        int32_t rc__ = enter_lane((ctx), (st), &(ctx)->last_sched, &(ctx)->has_last_sched);  \
        if (rc__ != EF_OK) return rc__;                                                       \
    } while (0)

// timing-enabled events are pooled: creating one costs microseconds, which is visible next to a 50 us decode wave
int32_t efk_timing_events(ef_ctx* ctx, cudaEvent_t* e0, cudaEvent_t* e1) {
    for (cudaEvent_t* e : {e0, e1}) {
        if (!ctx->timing_pool.empty()) {
            *e = ctx->timing_pool.back();
            ctx->timing_pool.pop_back();
        } else {
            EF_CUDA(ctx, cudaEventCreate(e));
        }
    }
    return EF_OK;
}

// ---------------------------------------------------------------------------------------------------
// lifetime
// ---------------------------------------------------------------------------------------------------
extern "C" int32_t ef_create(const ef_config* cfg, ef_ctx** out) {
    if (out) *out = nullptr;
    if (!cfg || !out) return ef_fail(nullptr, EF_ERR_INVALID_ARG, "ef_create: null argument");
    const ef_config& c = *cfg;
    if (c.n_layers < 1 || c.n_experts < 1 || c.top_k < 1 || c.d_model < 1 || c.d_ff < 1 || c.n_slots < 1 ||
        c.n_shared < 0 || c.max_tokens < 1 || c.device < 0)
        return ef_fail(nullptr, EF_ERR_INVALID_ARG, "ef_create: non-positive field in ef_config");
    if (c.expert_kind != 0 && c.expert_kind != 1)
        return ef_fail(nullptr, EF_ERR_INVALID_ARG, "ef_create: expert_kind must be 0 (SwiGLU) or 1 (ReLU)");
    if (c.d_model % 64 || c.d_ff % 128 || c.top_k > 8 || c.top_k > c.n_experts || c.n_experts > 256)
        return ef_fail(nullptr, EF_ERR_UNSUPPORTED,
                       "ef_create: need d_model%%64==0, d_ff%%128==0, top_k<=8, top_k<=n_experts<=256");
    ef_ctx* ctx = new ef_ctx();
    ctx->cfg = c;
    ctx->W = (int64_t)(c.expert_kind == 1 ? 2 : 3) * c.d_model * c.d_ff * 2;
    auto bail = [&](int32_t code, const char* what, cudaError_t e) {
        ef_fail(nullptr, code, "ef_create: %s: %s", what, cudaGetErrorString(e));
        ef_destroy(ctx);
        return code;
    };
    cudaError_t e;
    if ((e = cudaSetDevice(c.device)) != cudaSuccess) return bail(EF_ERR_CUDA, "cudaSetDevice", e);
    int sms = 0;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c.device)) != cudaSuccess)
        return bail(EF_ERR_CUDA, "cudaDeviceGetAttribute", e);
    ctx->n_sms = sms;
    ctx->n_arena_slots = c.n_slots + c.n_layers * c.n_shared;
    if ((e = cudaMalloc(&ctx->arena, (size_t)ctx->n_arena_slots * ctx->W)) != cudaSuccess)
        return bail(EF_ERR_OOM, "slot arena", e);
    ctx->h_rows = (int64_t)c.max_tokens * (c.top_k + c.n_shared);
    if ((e = cudaMalloc(&ctx->h_ws, (size_t)ctx->h_rows * c.d_ff * 2)) != cudaSuccess)
        return bail(EF_ERR_OOM, "h workspace", e);
    if ((e = cudaHostAlloc((void**)&ctx->counts_pinned, sizeof(int32_t) * (c.n_experts + 1), cudaHostAllocDefault)) !=
        cudaSuccess)
        return bail(EF_ERR_OOM, "pinned counts", e);
    if ((e = cudaEventCreateWithFlags(&ctx->counts_event, cudaEventDisableTiming)) != cudaSuccess)
        return bail(EF_ERR_CUDA, "event", e);
    if ((e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking)) != cudaSuccess)
        return bail(EF_ERR_CUDA, "copy stream", e);
    memset(ctx->counts_pinned, 0, sizeof(int32_t) * (c.n_experts + 1));
    ctx->ev_ring.resize(kRing, nullptr);
    ctx->ev_gen.assign(kRing, 0);
    for (int i = 0; i < kRing; ++i)
        if ((e = cudaEventCreateWithFlags(&ctx->ev_ring[i], cudaEventDisableTiming)) != cudaSuccess)
            return bail(EF_ERR_CUDA, "event ring", e);
    ctx->host_expert.assign((size_t)c.n_layers * c.n_experts, nullptr);
    ctx->host_owned.assign((size_t)c.n_layers * c.n_experts, 0);
    ctx->host_aliases.assign((size_t)c.n_layers * c.n_experts, 0);
    ctx->alias_src.assign((size_t)c.n_layers * c.n_experts, -1);
    ctx->shared_registered.assign((size_t)c.n_layers * std::max(1, c.n_shared), 0);
    ctx->slots.assign(c.n_slots, EfSlot());
    ctx->slot_of.assign((size_t)c.n_layers * c.n_experts, -1);
    ctx->phys.assign(c.n_slots, EfPhys());
    // early hand-back of a slot from inside a wave (run_wave): a device word and the driver's stream wait on it; without
    // the entry point the first-victim hit simply keeps running as a wave of its own
    {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuStreamWaitValue32", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess && fn) {
            if ((e = cudaMalloc((void**)&ctx->early_flag, 256)) != cudaSuccess) return bail(EF_ERR_OOM, "early-release word", e);
            if ((e = cudaMemset(ctx->early_flag, 0, 256)) != cudaSuccess) return bail(EF_ERR_CUDA, "early-release word", e);
            ctx->wait_value_fn = fn;
        }
    }
    efk_token_sched_static_init(ctx);      // ef_path_hamming_static's scratch address; never fails ef_create
    int32_t rc = efk_ffn_tc_init(ctx);
    if (rc != EF_OK) {
        g_create_err = "ef_create: " + ctx->err;
        ef_destroy(ctx);
        return rc;
    }
    *out = ctx;
    return EF_OK;
}

extern "C" int32_t ef_destroy(ef_ctx* ctx) {
    if (!ctx) return EF_OK;
    cudaSetDevice(ctx->cfg.device);
    cudaDeviceSynchronize();
    for (auto& sp : ctx->copy_spans) { cudaEventDestroy(sp.first); cudaEventDestroy(sp.second); }
    for (auto& k : ctx->kspans) { cudaEventDestroy(k.e0); cudaEventDestroy(k.e1); }
    for (auto ev : ctx->timing_pool) cudaEventDestroy(ev);
    for (auto ev : ctx->ev_ring) if (ev) cudaEventDestroy(ev);
    if (ctx->counts_event) cudaEventDestroy(ctx->counts_event);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    for (size_t i = 0; i < ctx->host_expert.size(); ++i)
        if (ctx->host_expert[i] && ctx->host_owned[i]) cudaFreeHost(ctx->host_expert[i]);
    if (ctx->counts_pinned) cudaFreeHost(ctx->counts_pinned);
    if (ctx->sched_words) cudaFree(ctx->sched_words);
    if (ctx->splitk_ws) cudaFree(ctx->splitk_ws);
    if (ctx->kprof1) cudaFree(ctx->kprof1);
    if (ctx->kprof2) cudaFree(ctx->kprof2);
    if (ctx->splitk_counters) cudaFree(ctx->splitk_counters);
    efk_token_sched_free(ctx);
    if (ctx->h_ws) cudaFree(ctx->h_ws);
    if (ctx->early_flag) cudaFree(ctx->early_flag);
    if (ctx->arena) cudaFree(ctx->arena);
    delete ctx;
    return EF_OK;
}

// pack (Wg, Wu, Wd) into the library layout (ef_internal.h): W13 rows interleaved by 128, every matrix tiled
static void pack_tiled(char* dst, int64_t rows, int64_t K, const char* (*src_row)(const void*, int64_t), const void* cookie) {
    const int64_t chunk = EF_ROWLET * 2;                     // one rowlet: 128 bytes
    for (int64_t r = 0; r < rows; ++r) {
        const char* src = src_row(cookie, r);
        char* d0 = dst + ef_tiled_index(r, 0, rows, K) * 2;
        const int64_t t = r / EF_TILE_ROWS;
        const int64_t h = std::min<int64_t>(EF_TILE_ROWS, rows - t * EF_TILE_ROWS);
        for (int64_t kb = 0; kb < K / EF_ROWLET; ++kb) memcpy(d0 + kb * h * chunk, src + kb * chunk, chunk);
    }
}

struct PackSrc { const char* a; const char* b; int64_t row_bytes; };

static void pack_expert(const ef_config& c, const void* wg, const void* wu, const void* wd, char* dst) {
    const int64_t d = c.d_model, f = c.d_ff;
    PackSrc down{(const char*)wd, nullptr, f * 2};
    auto plain = [](const void* ck, int64_t r) -> const char* {
        const PackSrc* p = (const PackSrc*)ck;
        return p->a + r * p->row_bytes;
    };
    if (c.expert_kind == 1) {              // non-gated: W1[f, d] then W2[d, f]
        PackSrc w1{(const char*)wg, nullptr, d * 2};
        pack_tiled(dst, f, d, plain, &w1);
        pack_tiled(dst + f * d * 2, d, f, plain, &down);
        return;
    }
    PackSrc w13{(const char*)wg, (const char*)wu, d * 2};
    auto interleaved = [](const void* ck, int64_t r) -> const char* {   // packed row r of W13
        const PackSrc* p = (const PackSrc*)ck;
        const int64_t j = r / (2 * EF_W13_BLOCK), i = r % (2 * EF_W13_BLOCK);
        return (i < EF_W13_BLOCK ? p->a + (j * EF_W13_BLOCK + i) * p->row_bytes
                                 : p->b + (j * EF_W13_BLOCK + i - EF_W13_BLOCK) * p->row_bytes);
    };
    pack_tiled(dst, 2 * f, d, interleaved, &w13);
    pack_tiled(dst + 2 * f * d * 2, d, f, plain, &down);
}

extern "C" int32_t ef_host_expert_register(ef_ctx* ctx, int32_t layer, int32_t expert, const void* w_gate,
                                           const void* w_up, const void* w_down) {
    EF_CHECK_CTX(ctx);
    const ef_config& c = ctx->cfg;
    if (c.expert_kind == 1 && w_up)
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_host_expert_register: w_up must be NULL for non-gated (ReLU) experts");
    if (!w_gate || (!w_up && c.expert_kind == 0) || !w_down || layer < 0 || layer >= c.n_layers || expert >= c.n_experts ||
        expert < -c.n_shared)
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_host_expert_register: bad layer/expert/pointer");
    EF_CUDA(ctx, cudaSetDevice(c.device));
    if (expert >= 0) {
        // re-registration replaces the packed host copy: not while another expert aliases it (the alias would dangle) and
        // not while a slot holds or is receiving the old weights (the hit would serve stale data, a copy in flight would
        // read freed pinned memory)
        const size_t g = (size_t)layer * c.n_experts + expert;
        if (ctx->host_expert[g] && ctx->host_aliases[g] > 0)
            return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_host_expert_register: (layer %d, expert %d) is aliased by %d other expert(s)",
                           layer, expert, ctx->host_aliases[g]);
        if (ctx->host_expert[g] && ctx->slot_of[g] >= 0)
            return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_host_expert_register: (layer %d, expert %d) is resident; ef_cache_evict it first",
                           layer, expert);
        if (ctx->host_expert[g]) EF_CUDA(ctx, cudaStreamSynchronize(ctx->copy_stream));   // an evicted expert's copy may still be in flight
    }
    void* buf = nullptr;
    cudaError_t e = cudaHostAlloc(&buf, (size_t)ctx->W, cudaHostAllocDefault);
    if (e != cudaSuccess) return ef_fail(ctx, EF_ERR_OOM, "pinned host pool: %s", cudaGetErrorString(e));
    pack_expert(c, w_gate, w_up, w_down, (char*)buf);
    if (expert >= 0) {
        size_t g = (size_t)layer * c.n_experts + expert;
        if (ctx->host_expert[g] && ctx->host_owned[g]) cudaFreeHost(ctx->host_expert[g]);
        else if (ctx->host_expert[g]) ctx->host_aliases[ctx->alias_src[g]]--;      // it was an alias until now
        ctx->host_expert[g] = buf;
        ctx->host_owned[g] = 1;
        return EF_OK;
    }
    const int s = -1 - expert;
    const int slot = c.n_slots + layer * c.n_shared + s;
    e = cudaMemcpy(ctx->arena + (size_t)slot * ctx->W, buf, (size_t)ctx->W, cudaMemcpyHostToDevice);
    cudaFreeHost(buf);
    if (e != cudaSuccess) { ctx->sticky = EF_ERR_CUDA; return ef_fail(ctx, EF_ERR_CUDA, "shared expert upload: %s", cudaGetErrorString(e)); }
    ctx->shared_registered[(size_t)layer * c.n_shared + s] = 1;
    return EF_OK;
}

extern "C" int32_t ef_host_expert_alias(ef_ctx* ctx, int32_t layer, int32_t expert, int32_t src_layer,
                                        int32_t src_expert) {
    EF_CHECK_CTX(ctx);
    const ef_config& c = ctx->cfg;
    if (layer < 0 || layer >= c.n_layers || expert < 0 || expert >= c.n_experts || src_layer < 0 ||
        src_layer >= c.n_layers || src_expert < 0 || src_expert >= c.n_experts)
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_host_expert_alias: bad ids");
    size_t g = (size_t)layer * c.n_experts + expert, sg = (size_t)src_layer * c.n_experts + src_expert;
    if (!ctx->host_expert[sg]) return ef_fail(ctx, EF_ERR_NOT_REGISTERED, "ef_host_expert_alias: source not registered");
    if (g == sg) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_host_expert_alias: an expert cannot alias itself");
    if (!ctx->host_owned[sg]) sg = (size_t)ctx->alias_src[sg];                    // alias of an alias: count on the owner
    if (ctx->host_expert[g]) {
        if (ctx->host_aliases[g] > 0 || ctx->slot_of[g] >= 0)
            return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_host_expert_alias: the target is aliased by others or resident");
        EF_CUDA(ctx, cudaStreamSynchronize(ctx->copy_stream));
        if (ctx->host_owned[g]) cudaFreeHost(ctx->host_expert[g]);
        else ctx->host_aliases[ctx->alias_src[g]]--;
    }
    ctx->host_expert[g] = ctx->host_expert[sg];
    ctx->host_owned[g] = 0;
    ctx->alias_src[g] = (int32_t)sg;
    ctx->host_aliases[sg]++;
    return EF_OK;
}

// ---------------------------------------------------------------------------------------------------
// thin wrappers around the memory-bound kernels
// ---------------------------------------------------------------------------------------------------
extern "C" int32_t ef_route_topk(ef_ctx* ctx, void* stream, const void* x, const void* w_router, const float* bias,
                                 int64_t bias_token_stride, int32_t T, int32_t renorm, int32_t* topk_idx,
                                 float* topk_w, float* logits_out) {
    EF_CHECK_CTX(ctx);
    if (T < 0 || (T > 0 && (!x || !w_router || !topk_idx || !topk_w)))
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_route_topk: null pointer or negative T");
    if (T > ctx->cfg.max_tokens) return ef_fail(ctx, EF_ERR_CAPACITY, "ef_route_topk: T > max_tokens");
    if (bias && bias_token_stride != 0 && bias_token_stride < ctx->cfg.n_experts)
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_route_topk: bias_token_stride must be 0 or >= E");
    EF_ENTER_LAYER(ctx, (cudaStream_t)stream);
    return efk_route_topk(ctx, (cudaStream_t)stream, x, w_router, bias, bias_token_stride, T, renorm ? 1 : 0,
                          topk_idx, topk_w, logits_out);
}

extern "C" int32_t ef_permute(ef_ctx* ctx, void* stream, const int32_t* topk_idx, const void* x, int32_t T,
                              void* x_perm, int32_t* counts, int32_t* offsets, int32_t* src, int32_t* inv,
                              int32_t* counts_host_pinned) {
    EF_CHECK_CTX(ctx);
    if (T < 0 || !counts || !offsets || (T > 0 && (!topk_idx || !x || !x_perm || !src || !inv)))
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_permute: null pointer or negative T");
    if (T > ctx->cfg.max_tokens) return ef_fail(ctx, EF_ERR_CAPACITY, "ef_permute: T > max_tokens");
    EF_ENTER_LAYER(ctx, (cudaStream_t)stream);
    int32_t* mirror = counts_host_pinned ? counts_host_pinned : ctx->counts_pinned;
    int32_t* err = ctx->counts_pinned + ctx->cfg.n_experts;
    *err = 0;
    int32_t rc = efk_permute(ctx, (cudaStream_t)stream, topk_idx, x, T, x_perm, counts, offsets, src, inv, mirror, err);
    if (rc != EF_OK) return rc;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing((cudaStream_t)stream, &cap) == cudaSuccess && cap == cudaStreamCaptureStatusActive) {
        ctx->counts_mirror = nullptr;  // captured into a graph: nothing has run, there is no mirror to wait for
        return EF_OK;
    }
    ctx->counts_mirror = mirror;       // what ef_expert_ffn_grouped(counts_host = NULL) reads once the event has fired
    EF_CUDA(ctx, cudaEventRecord(ctx->counts_event, (cudaStream_t)stream));
    return EF_OK;
}

extern "C" int32_t ef_combine(ef_ctx* ctx, void* stream, const void* y_perm, const int32_t* inv, const float* topk_w,
                              int32_t T, const void* residual, const void* y_shared, void* out) {
    EF_CHECK_CTX(ctx);
    if (T < 0 || (T > 0 && (!y_perm || !inv || !topk_w || !out)))
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_combine: null pointer or negative T");
    if (y_shared && ctx->cfg.n_shared == 0) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_combine: y_shared given but n_shared == 0");
    EF_ENTER_LAYER(ctx, (cudaStream_t)stream);
    return efk_combine(ctx, (cudaStream_t)stream, y_perm, inv, topk_w, T, residual, y_shared, out);
}

extern "C" int32_t ef_rmsnorm(ef_ctx* ctx, void* stream, const void* x, int32_t T, float eps, void* out) {
    EF_CHECK_CTX(ctx);
    if (T < 0 || (T > 0 && (!x || !out))) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_rmsnorm: null pointer or negative T");
    EF_ENTER_LAYER(ctx, (cudaStream_t)stream);
    return efk_rmsnorm(ctx, (cudaStream_t)stream, x, T, eps, out);
}

// ---------------------------------------------------------------------------------------------------
// cache policy
// ---------------------------------------------------------------------------------------------------
namespace {

inline bool pending(const EfSlot& s) { return s.pred_for != -1 && !s.used; }

int64_t next_visit_of_layer(int L, int layer, int64_t v) {
    const int64_t v1 = v + 1;
    int64_t r = (layer - v1) % L;
    if (r < 0) r += L;
    return v1 + r;
}

// first visit > v of the expert's layer where it is predicted active; visits without a supplied
// prediction count as "assume used"
int64_t est_next_use(ef_ctx* ctx, int32_t g, int64_t v) {
    const int E = ctx->cfg.n_experts, L = ctx->cfg.n_layers;
    const int layer = g / E, e = g % E;
    int64_t t = next_visit_of_layer(L, layer, v);
    for (;;) {
        auto it = ctx->pred.find(t);
        if (it == ctx->pred.end() || it->second[e]) return t;
        t += L;
    }
}

// class 0 empty; 1 mis-prefetched; 2 completed & next use later than target; 3 (on demand only) the rest
// Baseline policies (ef_set_cache_policy): least-recently-used over the whole pool, or over the
// requesting layer's own share of it (slots [layer * S / L, (layer + 1) * S / L)).  Empty slots first, then the smallest
// stamp; locked slots (this visit's experts) are skipped.  No predictions are consulted.
int pick_victim_lru(ef_ctx* ctx, int layer, const std::vector<char>& locked) {
    int s0 = 0, s1 = ctx->cfg.n_slots;
    if (ctx->policy == EF_POLICY_LAYER_LRU) {
        const int share = ctx->cfg.n_slots / ctx->cfg.n_layers;
        s0 = layer * share;
        s1 = s0 + share;
    }
    int best = -1;
    for (int s = s0; s < s1; ++s) {
        const EfSlot& sl = ctx->slots[s];
        if (sl.expert < 0) return s;
        if (locked[s]) continue;
        if (best < 0 || sl.stamp < ctx->slots[best].stamp) best = s;
    }
    return best;
}

int pick_victim(ef_ctx* ctx, int64_t v_now, int64_t target, bool allow3, const std::vector<char>& locked) {
    if (ctx->policy != EF_POLICY_PLEC) return pick_victim_lru(ctx, (int)(target % ctx->cfg.n_layers), locked);
    typedef std::tuple<int, int64_t, uint64_t, int> Key;
    bool have = false;
    Key best;
    for (int s = 0; s < ctx->cfg.n_slots; ++s) {
        const EfSlot& sl = ctx->slots[s];
        Key key;
        if (sl.expert < 0) {
            key = Key(0, 0, 0, s);
        } else if (locked[s]) {
            continue;
        } else if (pending(sl) && sl.pred_for <= v_now) {
            key = Key(1, 0, sl.stamp, s);
        } else {
            const int64_t nu = est_next_use(ctx, sl.expert, v_now);
            if (!pending(sl) && nu > target) key = Key(2, -nu, sl.stamp, s);
            else if (allow3) key = Key(3, -nu, sl.stamp, s);
            else continue;
        }
        if (!have || key < best) { best = key; have = true; }
    }
    return have ? std::get<3>(best) : -1;
}

void drain_copy_spans(ef_ctx* ctx, bool wait, float* acc_ms);

// policy bookkeeping of one load (slot table, counters): decided in policy order, at once
int32_t policy_load(ef_ctx* ctx, int slot, int32_t g, int64_t pred_for) {
    if (!ctx->host_expert[g])
        return ef_fail(ctx, EF_ERR_NOT_REGISTERED, "expert (layer %d, id %d) was never registered", g / ctx->cfg.n_experts,
                       g % ctx->cfg.n_experts);
    EfSlot& sl = ctx->slots[slot];
    if (sl.expert >= 0) {
        ctx->stats.evictions++;
        if (pending(sl)) ctx->stats.prefetch_wasted++;
        ctx->slot_of[sl.expert] = -1;
    }
    sl.expert = g;
    sl.pred_for = pred_for;
    sl.used = false;
    sl.stamp = ++ctx->tick;
    ctx->slot_of[g] = slot;
    ctx->stats.bytes_h2d += (uint64_t)ctx->W;
    return EF_OK;
}

// the physical H2D of one load: waits (on the copy stream) for the last wave that read the slot, then copies
int32_t enqueue_copy(ef_ctx* ctx, int slot, int32_t g) {
    EfPhys& ph = ctx->phys[slot];
    if (ph.has_flag) {
        // the slot's last reader hands it back from inside its launch: wait for the device word, not for the launch's end
        typedef CUresult (*WaitValueFn)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
        CUresult r = ((WaitValueFn)ctx->wait_value_fn)((CUstream)ctx->copy_stream, (CUdeviceptr)(uintptr_t)ctx->early_flag, ph.flag_target,
                                                       CU_STREAM_WAIT_VALUE_GEQ);
        if (r != CUDA_SUCCESS) return ef_fail(ctx, EF_ERR_CUDA, "cuStreamWaitValue32 failed: %d", (int)r);
        ph.has_flag = false;
    } else {
        EF_CUDA(ctx, ring_wait(ctx, ctx->copy_stream, ph.free_, ctx->last_compute, ctx->has_last_compute));
    }
    cudaEvent_t t0, t1;
    if (ctx->copy_spans.size() > 1024) drain_copy_spans(ctx, false, nullptr);
    {
        int32_t rc = efk_timing_events(ctx, &t0, &t1);
        if (rc != EF_OK) return rc;
    }
    EF_CUDA(ctx, cudaEventRecord(t0, ctx->copy_stream));
    // Finer-grained streaming: a large expert travels as two copies -- the first-GEMM weights
    // (packed W13, or W1), then Wd -- with a "ready" event after each, so GEMM1 of the visit's last wave runs while Wd is
    // still on the link.  Small experts travel whole (the gap between two copies would cost more link time than the
    // overlap wins).
    char* dst = ctx->arena + (size_t)slot * ctx->W;
    const char* srcp = (const char*)ctx->host_expert[g];
    const size_t w1_bytes = (size_t)(ctx->cfg.expert_kind == 1 ? 1 : 2) * ctx->cfg.d_model * ctx->cfg.d_ff * 2;
    cudaError_t e;
    ph.ready1 = EvHandle();
    if (ctx->chunk_min_bytes > 0 && ctx->W >= ctx->chunk_min_bytes) {
        EF_CUDA(ctx, cudaMemcpyAsync(dst, srcp, w1_bytes, cudaMemcpyHostToDevice, ctx->copy_stream));
        ph.ready1 = ring_record(ctx, ctx->copy_stream, &e);
        EF_CUDA(ctx, e);
        EF_CUDA(ctx, cudaMemcpyAsync(dst + w1_bytes, srcp + w1_bytes, (size_t)ctx->W - w1_bytes, cudaMemcpyHostToDevice,
                                     ctx->copy_stream));
    } else {
        EF_CUDA(ctx, cudaMemcpyAsync(dst, srcp, (size_t)ctx->W, cudaMemcpyHostToDevice, ctx->copy_stream));
    }
    EF_CUDA(ctx, cudaEventRecord(t1, ctx->copy_stream));
    ctx->copy_spans.emplace_back(t0, t1);
    ph.ready = ring_record(ctx, ctx->copy_stream, &e);
    EF_CUDA(ctx, e);
    ph.free_ = EvHandle();
    ph.waited_mask = 0;
    ph.waited = nullptr;
    return EF_OK;
}

int32_t issue_load(ef_ctx* ctx, int slot, int32_t g, int64_t pred_for) {
    int32_t rc = policy_load(ctx, slot, g, pred_for);
    return rc != EF_OK ? rc : enqueue_copy(ctx, slot, g);
}

void drain_copy_spans(ef_ctx* ctx, bool wait, float* acc_ms) {
    (void)acc_ms;
    auto& v = ctx->copy_spans;
    size_t keep = 0;
    for (size_t i = 0; i < v.size(); ++i) {
        bool done = wait ? (cudaEventSynchronize(v[i].second) == cudaSuccess)
                         : (cudaEventQuery(v[i].second) == cudaSuccess);
        if (done) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, v[i].first, v[i].second) == cudaSuccess) ctx->copy_ms += ms;
            ctx->timing_pool.push_back(v[i].first);
            ctx->timing_pool.push_back(v[i].second);
        } else {
            v[keep++] = v[i];
        }
    }
    v.resize(keep);
}

// one wave: groups (expert-local id e, slot) computed by one grouped launch (chunks of EF_MAX_GROUPS)
struct WaveItem { int32_t row0, rows, slot; };

// make `st` wait for the parts of the slot's expert that GEMM `which` (1 or 2) reads
int32_t wait_slot_ready(ef_ctx* ctx, cudaStream_t st, EfPhys& ph, int which) {
    if (ph.waited != st) { ph.waited = st; ph.waited_mask = 0; }
    if (which == 1 && ph.ready1.idx >= 0) {
        if (!(ph.waited_mask & 1)) {
            EF_CUDA(ctx, ring_wait(ctx, st, ph.ready1, ctx->copy_stream));
            ph.waited_mask |= 1;
        }
        return EF_OK;
    }
    if (ph.ready.idx >= 0 && !(ph.waited_mask & 2)) {
        EF_CUDA(ctx, ring_wait(ctx, st, ph.ready, ctx->copy_stream));
        ph.waited_mask |= 3;      // the whole-expert event is recorded after the first-chunk event
    }
    return EF_OK;
}

// One wave.  Normally ONE launch that runs both GEMMs (ffn_tc.cu) once every member's weights have landed.  Only the
// LAST wave of a visit may run as two launches when its expert is still arriving in two chunks: GEMM1 is gated on the
// first chunk (W13 / W1) and overlaps the transfer of Wd, so the tail of the visit after its final copy is one GEMM2.  For
// every earlier wave that overlap buys nothing -- the next wave's copies are on the link anyway -- and one launch is faster.
// early_slot >= 0: that member's slot is about to be overwritten by a copy that is enqueued right after this wave; it goes
// first in the wave's table and, if the wave's tiling allows (efk_ffn_tc), is handed back from inside the launch.
int32_t run_wave(ef_ctx* ctx, cudaStream_t st, const void* x_perm, void* y_perm, const std::vector<WaveItem>& items_in,
                 bool last_of_visit = false, int early_slot = -1) {
    if (items_in.empty()) return EF_OK;
    std::vector<WaveItem> items = items_in;
    if (early_slot >= 0)
        std::stable_partition(items.begin(), items.end(), [&](const WaveItem& it) { return it.slot == early_slot; });
    auto& phys = ctx->phys;
    int32_t rc;
    bool two_launches = !ctx->fused_waves;
    if (last_of_visit)
        for (const WaveItem& it : items) {
            const EfPhys& ph = phys[it.slot];
            if (ph.ready1.idx >= 0 && !(ph.waited == st && (ph.waited_mask & 2))) two_launches = true;
        }
    auto launch = [&](int phase) -> int32_t {
        for (size_t base = 0; base < items.size(); base += EF_MAX_GROUPS) {
            EfWaveTable tab;
            tab.n = (int32_t)std::min<size_t>(EF_MAX_GROUPS, items.size() - base);
            for (int i = 0; i < tab.n; ++i) {
                const WaveItem& it = items[base + i];
                tab.g[i] = EfWaveGroup{it.row0, it.row0, it.row0, it.rows, it.slot};
            }
            EfEarly early;
            early.want = early_slot >= 0 && base == 0 && phase == 3 && tab.g[0].slot == early_slot;
            int32_t r = efk_ffn_grouped(ctx, st, x_perm, y_perm, tab, phase, &early);
            if (r != EF_OK) return r;
            if (early.used) {
                ctx->early_target += early.add;
                phys[early_slot].has_flag = true;
                phys[early_slot].flag_target = ctx->early_target;
            }
        }
        return EF_OK;
    };
    if (two_launches) {
        for (int which = 1; which <= 2; ++which) {
            for (const WaveItem& it : items)
                if ((rc = wait_slot_ready(ctx, st, phys[it.slot], which)) != EF_OK) return rc;
            if ((rc = launch(which)) != EF_OK) return rc;
        }
    } else {
        for (const WaveItem& it : items)
            if ((rc = wait_slot_ready(ctx, st, phys[it.slot], 2)) != EF_OK) return rc;
        if ((rc = launch(3)) != EF_OK) return rc;
    }
    cudaError_t e;
    EvHandle ev = ring_record(ctx, st, &e);
    EF_CUDA(ctx, e);
    for (const WaveItem& it : items) {
        phys[it.slot].free_ = ev;
        if (it.slot != early_slot) phys[it.slot].has_flag = false;
    }
    return EF_OK;
}

// would run_wave(items, false, early_slot) hand that slot back from inside its launch?
bool wave_can_release_early(ef_ctx* ctx, cudaStream_t st, const void* x_perm, void* y_perm, const std::vector<WaveItem>& items_in, int early_slot) {
    if (!ctx->early_release || !ctx->fused_waves || !ctx->early_flag || !ctx->wait_value_fn || items_in.size() > (size_t)EF_MAX_GROUPS) return false;
#ifdef EF_DIAG
    if (ctx->debug_simt) return false;
#endif
    std::vector<WaveItem> items = items_in;
    std::stable_partition(items.begin(), items.end(), [&](const WaveItem& it) { return it.slot == early_slot; });
    EfWaveTable tab;
    tab.n = (int32_t)items.size();
    for (int i = 0; i < tab.n; ++i) tab.g[i] = EfWaveGroup{items[i].row0, items[i].row0, items[i].row0, items[i].rows, items[i].slot};
    EfEarly q;
    q.want = true;
    q.dry = true;
    return efk_ffn_tc(ctx, st, x_perm, y_perm, tab, 3, &q) == EF_OK && q.used;
}

// Miss waves.  Every on-demand expert could be its own wave (compute starts the moment its copy lands), but for small
// experts that is one launch per ~0.3 ms copy, each far too short to fill the GPU.  The batcher groups consecutive
// misses into waves: never less than ~wave_bytes of link traffic per wave, and -- while many misses are still to come --
// HALF of what is left (a visit with 40 small misses runs them as waves of 20, 10 and 10 experts): the big early
// waves are real grouped GEMMs, each finishes long before the next, smaller wave's copies have landed.  When an expert is
// large enough to be copied in two chunks (>= chunk_min_bytes: its FFN is a good fraction of a millisecond) the last miss
// of a visit is a wave of its own, so the tail after the final copy is one expert's GEMM2; for small experts the last
// misses stay together -- a launch per 17 MB expert costs more in ramp and tail than the others add to the wave.
// Physical scheduling only: which slot a miss takes and every counter were decided before the item got here.
struct MissBatcher {
    ef_ctx* ctx; cudaStream_t st; const void* x_perm; void* y_perm;
    std::vector<WaveItem> open;
    int min_wave;           // experts per wave from wave_bytes
    int remaining;          // misses of this visit not yet pushed (set by the caller)
    int target;             // size of the wave being collected
    MissBatcher(ef_ctx* c, cudaStream_t s, const void* x, void* y, int n_misses)
        : ctx(c), st(s), x_perm(x), y_perm(y), remaining(n_misses) {
        min_wave = (int)std::max<int64_t>(1, std::min<int64_t>(EF_MAX_GROUPS, ctx->wave_bytes / ctx->W));
        slot_wave.assign(ctx->cfg.n_slots, 0);
        target = next_target();
    }
    int next_target() const {
        if (ctx->wave_bytes == 0) return 1;
        int t = std::min(EF_MAX_GROUPS, std::max(min_wave, remaining / 2));
        // small experts: no trailing wave of one or two -- what is left joins this wave (see push)
        if (!last_alone() && remaining - t <= std::max(2, min_wave / 2) && remaining <= EF_MAX_GROUPS) t = std::max(t, remaining);
        return t;
    }
    bool last_alone() const { return ctx->chunk_min_bytes > 0 && ctx->W >= ctx->chunk_min_bytes; }
    bool holds_slot(int slot) const {
        for (const WaveItem& it : open) if (it.slot == slot) return true;
        return false;
    }
    std::vector<int> slot_wave;   // per slot: sequence number of the miss wave that read it last (0: none of them)
    int seq = 1;
    int32_t flush(bool last_of_visit = false) {
        if (open.empty()) return EF_OK;
        for (const WaveItem& it : open) slot_wave[it.slot] = seq;
        ++seq;
        int32_t rc = run_wave(ctx, st, x_perm, y_perm, open, last_of_visit);
        open.clear();
        target = next_target();
        return rc;
    }
    int32_t push(const WaveItem& it, bool last_of_visit) {
        int32_t rc = EF_OK;
        if (last_of_visit && last_alone() && !open.empty() && (rc = flush()) != EF_OK) return rc;
        open.push_back(it);
        --remaining;
        if ((int)open.size() >= target || last_of_visit) rc = flush(last_of_visit);
        return rc;
    }
};

}  // namespace

int32_t efk_ffn_grouped(ef_ctx* ctx, cudaStream_t st, const void* x, void* y, const EfWaveTable& tab, int phase, EfEarly* early) {
#ifdef EF_DIAG
    if (ctx->debug_simt) return efk_ffn_simt(ctx, st, x, y, tab, phase);     // bring-up aid, diag library only (ef_diag.h)
#endif
    return efk_ffn_tc(ctx, st, x, y, tab, phase, early);
}

extern "C" int32_t ef_expert_ffn_grouped(ef_ctx* ctx, void* stream, int64_t visit, int32_t layer, const void* x_perm,
                                         const int32_t* counts_host, void* y_perm) {
    EF_CHECK_CTX(ctx);
    const ef_config& c = ctx->cfg;
    cudaStream_t st = (cudaStream_t)stream;
    if (layer < 0 || layer >= c.n_layers || !x_perm || !y_perm)
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_expert_ffn_grouped: bad layer or null pointer");
    if (visit < 0 || (int32_t)(visit % c.n_layers) != layer)
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_expert_ffn_grouped: visit %% n_layers must equal layer");
    if (!counts_host) {
        if (!ctx->counts_mirror) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_expert_ffn_grouped: counts_host is NULL and no ef_permute has run");
        EF_CUDA(ctx, cudaEventSynchronize(ctx->counts_event));   // the one device->host sync per visit
        counts_host = ctx->counts_mirror;
        if (ctx->counts_pinned[c.n_experts])
            return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_expert_ffn_grouped: the last ef_permute saw top-k indices outside [0, n_experts)");
    }
    const int E = c.n_experts;
    std::vector<int32_t> off(E + 1, 0);
    for (int e = 0; e < E; ++e) {
        if (counts_host[e] < 0) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_expert_ffn_grouped: negative count");
        off[e + 1] = off[e] + counts_host[e];
    }
    if ((int64_t)off[E] > (int64_t)c.max_tokens * c.top_k)
        return ef_fail(ctx, EF_ERR_CAPACITY, "ef_expert_ffn_grouped: sum(counts) > max_tokens * top_k");
    EF_ENTER_LAYER(ctx, st);

    // lookup (R6)
    std::vector<int> hits, misses;
    for (int e = 0; e < E; ++e) {
        if (counts_host[e] == 0) continue;
        (ctx->slot_of[(size_t)layer * E + e] >= 0 ? hits : misses).push_back(e);
    }
    ctx->stats.lookups += hits.size() + misses.size();
    ctx->stats.hits += hits.size();
    ctx->stats.misses += misses.size();
    std::vector<char> locked(c.n_slots, 0);
    std::vector<WaveItem> wave0;
    for (int e : hits) {
        const int s = ctx->slot_of[(size_t)layer * E + e];
        EfSlot& sl = ctx->slots[s];
        if (pending(sl)) ctx->stats.prefetch_used++;
        sl.used = true;
        sl.stamp = ++ctx->tick;
        locked[s] = 1;
        wave0.push_back(WaveItem{off[e], counts_host[e], s});
    }
    // ---- policy, in policy order (R12: ascending expert id), all of it before anything physical: every decision depends
    // on the slot table alone ("completed" = enqueued, R9)
    struct Miss { WaveItem item; int32_t g; int gen; };     // gen: 0 = the victim slot held nothing of this visit's misses
    std::vector<Miss> planA, planB;
    std::vector<int> gen_of_slot(c.n_slots, -1);
    // phase A: on-demand loads into empty / mis-prefetched / completed slots; their copies overlap wave 0
    std::vector<int> rest;
    for (int e : misses) {
        const int s = pick_victim(ctx, visit, visit, false, locked);
        if (s < 0) { rest.push_back(e); continue; }
        int32_t rc = policy_load(ctx, s, layer * E + e, -1);
        if (rc != EF_OK) return rc;
        ctx->stats.ondemand_loads++;
        ctx->slots[s].used = true;
        locked[s] = 1;
        gen_of_slot[s] = 0;
        planA.push_back(Miss{WaveItem{off[e], counts_host[e], s}, layer * E + e, 0});
    }
    // phase B: the pool was full of this visit's own experts and useful prefetches; the locks drop, and each remaining
    // miss takes a class 0-3 victim -- now including this visit's hits and the misses that came before it
    std::fill(locked.begin(), locked.end(), 0);
    for (int e : rest) {
        const int s = pick_victim(ctx, visit, visit, true, locked);
        if (s < 0) return ef_fail(ctx, EF_ERR_CAPACITY, "ef_expert_ffn_grouped: no victim slot (internal)");
        int32_t rc = policy_load(ctx, s, layer * E + e, -1);
        if (rc != EF_OK) return rc;
        ctx->stats.ondemand_loads++;
        ctx->slots[s].used = true;
        const int gen = gen_of_slot[s] < 0 ? 0 : gen_of_slot[s] + 1;
        gen_of_slot[s] = gen;
        planB.push_back(Miss{WaveItem{off[e], counts_host[e], s}, layer * E + e, gen});
    }
    // ---- physical order of the copies (never part of the policy; EF_OPT_COPY_ORDER): misses that do not
    // wait for one another go on the link with the most routed rows first -- the largest GEMMs start earliest and the
    // visit's tail after its final copy is its smallest expert -- and a miss that reuses the slot of an earlier miss of
    // this visit (a later "generation") follows the generation it waits for.
    if (ctx->copy_order == 1) {
        auto more_rows = [](const Miss& a, const Miss& b) { return a.item.rows > b.item.rows; };
        std::stable_sort(planA.begin(), planA.end(), more_rows);
        std::stable_sort(planB.begin(), planB.end(), [](const Miss& a, const Miss& b) {
            return a.gen != b.gen ? a.gen < b.gen : a.item.rows > b.item.rows;
        });
    }
    int32_t rc = EF_OK;
    for (const Miss& m : planA)
        if ((rc = enqueue_copy(ctx, m.item.slot, m.g)) != EF_OK) return rc;
    // Wave 0 = the hits.  The first phase-B copy is about to overwrite the slot of one of these very hits, and it waits
    // for the "free" event of the wave that read the slot.  Copies are far slower than waves, so only the FIRST one
    // matters: that hit runs as its own wave first, so the copy starts after one expert's FFN instead of after the whole
    // wave (physical ordering only: the policy and its accounting are unchanged).
    int first_victim = (!planB.empty() && wave0.size() > 1) ? planB[0].item.slot : -1;
    size_t split_at = wave0.size();
    for (size_t i = 0; i < wave0.size(); ++i)
        if (wave0[i].slot == first_victim) split_at = i;
    const bool no_misses = planA.empty() && planB.empty();
    if (split_at == wave0.size()) {
        rc = run_wave(ctx, st, x_perm, y_perm, wave0, no_misses);
        if (rc != EF_OK) return rc;
    } else {
        if (wave_can_release_early(ctx, st, x_perm, y_perm, wave0, first_victim)) {
            // ONE wave: the first victim's units are ticketed first and hand its slot back from inside the launch
            // (EF_OPT_EARLY_RELEASE; the copy waits on a device word instead of on an event behind a launch of its own)
            rc = run_wave(ctx, st, x_perm, y_perm, wave0, false, first_victim);
            if (rc != EF_OK) return rc;
        } else {
            std::vector<WaveItem> others;
            for (size_t i = 0; i < wave0.size(); ++i)
                if (i != split_at) others.push_back(wave0[i]);
            rc = run_wave(ctx, st, x_perm, y_perm, std::vector<WaveItem>{wave0[split_at]});
            if (rc != EF_OK) return rc;
            rc = run_wave(ctx, st, x_perm, y_perm, others);
            if (rc != EF_OK) return rc;
        }
    }
    MissBatcher mb(ctx, st, x_perm, y_perm, (int)(planA.size() + planB.size()));
    for (size_t i = 0; i < planA.size(); ++i)   // compute starts as the copies land, one grouped launch per batch
        if ((rc = mb.push(planA[i].item, planB.empty() && i + 1 == planA.size())) != EF_OK) return rc;
    // The copy into a slot waits for the "free" event of the wave that read the slot last: that wave must be enqueued first.
    // A miss whose slot belongs to a member of the OPEN wave therefore steps back behind the misses that can go now
    // (EF_OPT_COPY_ORDER = 1; in policy copy order the open wave is launched early instead, as a small wave of its own): the
    // link stays busy, and the open wave fills up to its target instead of being flushed with a handful of experts.  A miss
    // never overtakes an earlier miss of the same slot (an earlier generation).  Among the misses that can go, the one
    // whose slot was read by the OLDEST wave goes first: the copy stream is a FIFO, and a copy that has to wait for a wave
    // that has only just been launched would hold up every copy behind it.
    std::vector<char> done(planB.size(), 0);
    size_t n_done = 0;
    while (n_done < planB.size()) {
        size_t pick = planB.size(), first_head = planB.size();
        for (size_t i = 0; i < planB.size(); ++i) {
            if (done[i]) continue;
            bool head = true;                         // planB is in generation order: an earlier entry of the same slot goes first
            for (size_t k = 0; k < i && head; ++k) head = done[k] || planB[k].item.slot != planB[i].item.slot;
            if (!head) continue;
            if (first_head == planB.size()) first_head = i;
            if (ctx->copy_order != 1) {               // policy copy order: no overtaking
                if (!mb.holds_slot(planB[i].item.slot)) pick = i;
                break;
            }
            if (mb.holds_slot(planB[i].item.slot)) continue;
            if (pick == planB.size() || mb.slot_wave[planB[i].item.slot] < mb.slot_wave[planB[pick].item.slot]) pick = i;
        }
        if (pick == planB.size()) {                   // whatever could go next waits for the open wave: launch it
            if ((rc = mb.flush()) != EF_OK) return rc;
            pick = first_head;
        }
        const Miss& m = planB[pick];
        if ((rc = enqueue_copy(ctx, m.item.slot, m.g)) != EF_OK) return rc;
        done[pick] = 1;
        ++n_done;
        if ((rc = mb.push(m.item, n_done == planB.size())) != EF_OK) return rc;
    }
    return mb.flush();
}

extern "C" int32_t ef_expert_ffn_grouped_resident(ef_ctx* ctx, void* stream, const void* x_perm, int32_t n_groups,
                                                  const int32_t* row_begin, const int32_t* rows,
                                                  const int32_t* slots, void* y_perm) {
    EF_CHECK_CTX(ctx);
    if (n_groups < 0 || (n_groups > 0 && (!x_perm || !y_perm || !row_begin || !rows || !slots)))
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_expert_ffn_grouped_resident: null pointer");
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<WaveItem> items;
    for (int i = 0; i < n_groups; ++i) {
        if (rows[i] == 0) continue;
        if (rows[i] < 0 || row_begin[i] < 0 || slots[i] < 0 || slots[i] >= ctx->cfg.n_slots ||
            (int64_t)row_begin[i] + rows[i] > (int64_t)ctx->cfg.max_tokens * ctx->cfg.top_k)
            return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_expert_ffn_grouped_resident: bad group %d", i);
        items.push_back(WaveItem{row_begin[i], rows[i], slots[i]});
    }
    EF_ENTER_LAYER(ctx, st);
    return run_wave(ctx, st, x_perm, y_perm, items);
}

extern "C" int32_t ef_shared_ffn(ef_ctx* ctx, void* stream, int32_t layer, const void* x, int32_t T, void* y_shared) {
    EF_CHECK_CTX(ctx);
    const ef_config& c = ctx->cfg;
    if (c.n_shared == 0) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_shared_ffn: n_shared == 0");
    if (layer < 0 || layer >= c.n_layers || T < 0 || (T > 0 && (!x || !y_shared)))
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_shared_ffn: bad argument");
    if (T > c.max_tokens) return ef_fail(ctx, EF_ERR_CAPACITY, "ef_shared_ffn: T > max_tokens");
    if (T == 0) return EF_OK;
    EfWaveTable tab;
    if (c.n_shared > EF_MAX_GROUPS) return ef_fail(ctx, EF_ERR_UNSUPPORTED, "ef_shared_ffn: too many shared experts");
    tab.n = c.n_shared;
    for (int s = 0; s < c.n_shared; ++s) {
        if (!ctx->shared_registered[(size_t)layer * c.n_shared + s])
            return ef_fail(ctx, EF_ERR_NOT_REGISTERED, "shared expert %d of layer %d not registered", s, layer);
        // every token goes through every shared expert; their h rows live behind the routed region of the workspace
        tab.g[s] = EfWaveGroup{0, c.max_tokens * c.top_k + s * c.max_tokens, s * T, T, c.n_slots + layer * c.n_shared + s};
    }
    EF_ENTER_LAYER(ctx, (cudaStream_t)stream);
    return efk_ffn_grouped(ctx, (cudaStream_t)stream, x, y_shared, tab, 3);
}

extern "C" int32_t ef_cache_prefetch(ef_ctx* ctx, int64_t visit_now, const uint8_t* predicted, int32_t n_ahead) {
    EF_CHECK_CTX(ctx);
    const ef_config& c = ctx->cfg;
    if (n_ahead < 0 || (n_ahead > 0 && !predicted) || visit_now < -1)
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_cache_prefetch: bad argument");
    const int E = c.n_experts, L = c.n_layers;
    if (ctx->policy != EF_POLICY_PLEC) return EF_OK;      // the LRU baselines neither predict nor prefetch
    for (int i = 0; i < n_ahead; ++i)
        ctx->pred[visit_now + 1 + i] = std::vector<uint8_t>(predicted + (size_t)i * E, predicted + (size_t)(i + 1) * E);
    while (!ctx->pred.empty() && ctx->pred.begin()->first <= visit_now) ctx->pred.erase(ctx->pred.begin());
    const int span = c.prefetch_horizon > 0 ? std::min(c.prefetch_horizon, n_ahead) : n_ahead;
    std::vector<char> no_lock(c.n_slots, 0);
    for (int64_t t = visit_now + 1; t <= visit_now + span; ++t) {
        const int layer = (int)(t % L);
        const std::vector<uint8_t>& p = ctx->pred[t];
        for (int e = 0; e < E; ++e) {
            if (!p[e]) continue;
            const int32_t g = layer * E + e;
            const int cur = ctx->slot_of[g];
            if (cur >= 0) {
                EfSlot& sl = ctx->slots[cur];
                if (pending(sl) && sl.pred_for <= visit_now) sl.pred_for = t;   // R25: re-target a stale prefetch
                continue;
            }
            const int s = pick_victim(ctx, visit_now, t, false, no_lock);
            if (s < 0) return EF_OK;   // pool is full of useful experts
            int32_t rc = issue_load(ctx, s, g, t);
            if (rc != EF_OK) return rc;
            ctx->stats.prefetch_issued++;
        }
    }
    return EF_OK;
}

extern "C" int32_t ef_cache_evict(ef_ctx* ctx, int32_t layer, const int32_t* experts, int32_t n) {
    EF_CHECK_CTX(ctx);
    const ef_config& c = ctx->cfg;
    if (layer < 0 || layer >= c.n_layers || n < 0 || (n > 0 && !experts))
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_cache_evict: bad argument");
    for (int i = 0; i < n; ++i) {
        if (experts[i] < 0 || experts[i] >= c.n_experts) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_cache_evict: bad expert id");
        const int32_t g = layer * c.n_experts + experts[i];
        const int s = ctx->slot_of[g];
        if (s < 0) continue;
        EfSlot& sl = ctx->slots[s];
        ctx->stats.evictions++;
        if (pending(sl)) ctx->stats.prefetch_wasted++;
        ctx->slot_of[g] = -1;
        sl.expert = -1; sl.pred_for = -1; sl.used = false; sl.stamp = 0;
    }
    return EF_OK;
}

extern "C" int32_t ef_token_schedule(ef_ctx* ctx, void* stream, const uint8_t* paths, int32_t N, int32_t LE, int32_t c0,
                                     int32_t c1, int32_t max_iter, int32_t* batch_of, int32_t* perm, int32_t* info,
                                     uint8_t* batch_paths) {
    EF_CHECK_CTX(ctx);
    if (!paths || !batch_of || !perm || !info) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_token_schedule: null pointer");
    if (N < 2 || (N & 1) || c0 < 0 || c1 < 0 || c0 >= N || c1 >= N || c0 == c1 || max_iter < 1 || LE < 1)
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_token_schedule: need even N >= 2, distinct centroids in [0, N), max_iter >= 1");
    if (N > EF_TS_MAX_TOKENS || LE > 32767 || max_iter > 64)
        return ef_fail(ctx, EF_ERR_UNSUPPORTED, "ef_token_schedule: N <= %d, LE <= 32767, max_iter <= 64", EF_TS_MAX_TOKENS);
    EF_ENTER_SCHED(ctx, (cudaStream_t)stream);
    return efk_token_schedule(ctx, (cudaStream_t)stream, paths, N, LE, c0, c1, max_iter, batch_of, perm, info, batch_paths);
}

extern "C" int32_t ef_reindex_rows(ef_ctx* ctx, void* stream, const void* src, const int32_t* perm, int32_t n_rows,
                                   int64_t row_bytes, void* dst) {
    EF_CHECK_CTX(ctx);
    if (n_rows < 0 || row_bytes < 0 || (n_rows > 0 && row_bytes > 0 && (!src || !perm || !dst)) || src == dst)
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_reindex_rows: bad argument (out of place only)");
    if ((row_bytes & 15) || ((uintptr_t)src & 15) || ((uintptr_t)dst & 15) || row_bytes / 16 > INT32_MAX)
        return ef_fail(ctx, EF_ERR_UNSUPPORTED, "ef_reindex_rows: rows must be multiples of 16 bytes, 16-byte aligned");
    if (n_rows == 0 || row_bytes == 0) return EF_OK;
    EF_ENTER_SCHED(ctx, (cudaStream_t)stream);
    return efk_reindex_rows(ctx, (cudaStream_t)stream, src, perm, n_rows, row_bytes, dst);
}

extern "C" int32_t ef_path_hamming(ef_ctx* ctx, void* stream, const uint8_t* paths, int32_t N, int32_t LE,
                                   uint16_t* dist_out) {
    EF_CHECK_CTX(ctx);
    if (N < 0 || (N > 0 && (!paths || !dist_out)) || LE < 1) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_path_hamming: bad argument");
    if (N > EF_TS_MAX_TOKENS || LE > 32767 || ((uintptr_t)dist_out & 15))
        return ef_fail(ctx, EF_ERR_UNSUPPORTED, "ef_path_hamming: N <= %d, LE <= 32767, dist_out 16-byte aligned", EF_TS_MAX_TOKENS);
    if (N == 0) return EF_OK;
    EF_ENTER_SCHED(ctx, (cudaStream_t)stream);
    return efk_path_hamming(ctx, (cudaStream_t)stream, paths, N, LE, dist_out);
}

extern "C" int32_t ef_path_hamming_static(ef_ctx* ctx, void* stream, const uint8_t* paths, int32_t N, int32_t LE,
                                          uint16_t* dist_out) {
    EF_CHECK_CTX(ctx);
    if (N < 0 || (N > 0 && (!paths || !dist_out)) || LE < 1) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_path_hamming_static: bad argument");
    if (N > EF_TS_MAX_TOKENS || LE > 32767 || ((uintptr_t)dist_out & 15))
        return ef_fail(ctx, EF_ERR_UNSUPPORTED, "ef_path_hamming_static: N <= %d, LE <= 32767, dist_out 16-byte aligned", EF_TS_MAX_TOKENS);
    if (N == 0) return EF_OK;
    EF_ENTER_SCHED(ctx, (cudaStream_t)stream);
    return efk_path_hamming_static(ctx, (cudaStream_t)stream, paths, N, LE, dist_out);
}

extern "C" int32_t ef_cache_get_stats(ef_ctx* ctx, ef_cache_stats* out) {
    EF_CHECK_CTX(ctx);
    if (!out) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_cache_get_stats: null");
    *out = ctx->stats;
    return EF_OK;
}

extern "C" int32_t ef_cache_reset_stats(ef_ctx* ctx) {
    EF_CHECK_CTX(ctx);
    ctx->stats = ef_cache_stats();
    drain_copy_spans(ctx, true, nullptr);
    ctx->copy_ms = 0.f;
    return EF_OK;
}

extern "C" int32_t ef_cache_snapshot(ef_ctx* ctx, int32_t* slot_to_expert) {
    EF_CHECK_CTX(ctx);
    if (!slot_to_expert) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_cache_snapshot: null");
    for (int s = 0; s < ctx->cfg.n_slots; ++s) slot_to_expert[s] = ctx->slots[s].expert;
    return EF_OK;
}

extern "C" int32_t ef_cache_clear(ef_ctx* ctx) {
    EF_CHECK_CTX(ctx);
    for (auto& sl : ctx->slots) { sl.expert = -1; sl.pred_for = -1; sl.used = false; sl.stamp = 0; }
    std::fill(ctx->slot_of.begin(), ctx->slot_of.end(), -1);
    ctx->pred.clear();
    ctx->tick = 0;
    return EF_OK;
}

extern "C" int32_t ef_copy_busy_ms(ef_ctx* ctx, float* ms_out) {
    EF_CHECK_CTX(ctx);
    if (!ms_out) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_copy_busy_ms: null");
    EF_CUDA(ctx, cudaStreamSynchronize(ctx->copy_stream));
    drain_copy_spans(ctx, true, nullptr);
    *ms_out = ctx->copy_ms;
    return EF_OK;
}

extern "C" int32_t ef_sync(ef_ctx* ctx) {
    EF_CHECK_CTX(ctx);
    EF_CUDA(ctx, cudaStreamSynchronize(ctx->copy_stream));
    EF_CUDA(ctx, cudaDeviceSynchronize());
    return EF_OK;
}

extern "C" const char* ef_last_error(ef_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

extern "C" int64_t ef_launch_count(ef_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int32_t ef_set_cache_policy(ef_ctx* ctx, int32_t policy) {
    EF_CHECK_CTX(ctx);
    if (policy != EF_POLICY_PLEC && policy != EF_POLICY_LRU && policy != EF_POLICY_LAYER_LRU)
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_set_cache_policy: unknown policy %d", policy);
    if (policy == EF_POLICY_LAYER_LRU && ctx->cfg.n_slots < ctx->cfg.n_layers)
        return ef_fail(ctx, EF_ERR_CAPACITY, "ef_set_cache_policy: per-layer LRU needs at least one slot per layer");
    for (const EfSlot& sl : ctx->slots)
        if (sl.expert >= 0) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_set_cache_policy: the slot table must be empty (ef_cache_clear)");
    ctx->policy = policy;
    return EF_OK;
}

extern "C" int32_t ef_set_option(ef_ctx* ctx, int32_t key, int64_t value) {
    EF_CHECK_CTX(ctx);
    switch (key) {
        case EF_OPT_SPLITK:
            if (value < 0 || value > 16) return ef_fail(ctx, EF_ERR_INVALID_ARG, "EF_OPT_SPLITK: 0 (auto), 1 (off) or 2..16");
            ctx->splitk_mode = (int32_t)value;
            return EF_OK;
        case EF_OPT_WAVE_BYTES:
            if (value < 0) return ef_fail(ctx, EF_ERR_INVALID_ARG, "EF_OPT_WAVE_BYTES: negative");
            ctx->wave_bytes = value;
            return EF_OK;
        case EF_OPT_CHUNK_MIN_BYTES:
            if (value < 0) return ef_fail(ctx, EF_ERR_INVALID_ARG, "EF_OPT_CHUNK_MIN_BYTES: negative");
            ctx->chunk_min_bytes = value;
            return EF_OK;
        case EF_OPT_FUSED_WAVES:
            ctx->fused_waves = value ? 1 : 0;
            return EF_OK;
        case EF_OPT_TOKEN_SCHED_PATH:
            ctx->ts_force_multi = value ? 1 : 0;
            return EF_OK;
        case EF_OPT_EARLY_RELEASE:
            ctx->early_release = value ? 1 : 0;
            return EF_OK;
        case EF_OPT_COPY_ORDER:
            if (value != 0 && value != 1) return ef_fail(ctx, EF_ERR_INVALID_ARG, "EF_OPT_COPY_ORDER: 0 (policy order) or 1 (most rows first)");
            ctx->copy_order = (int32_t)value;
            return EF_OK;
        default:
            return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_set_option: unknown key %d", key);
    }
}

// wait for the recorded launch spans, fold them into the totals and the per-launch log, recycle their events
static void drain_kernel_spans(ef_ctx* ctx) {
    for (auto& k : ctx->kspans) {
        cudaEventSynchronize(k.e1);
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, k.e0, k.e1) == cudaSuccess) {
            ef_kernel_times& t = ctx->ktimes;
            if (k.which == 1) { t.gemm1_ms += ms; t.gemm1_launches++; t.gemm1_rows += k.rows; t.gemm1_groups += k.groups; }
            else if (k.which == 2) { t.gemm2_ms += ms; t.gemm2_launches++; t.gemm2_rows += k.rows; t.gemm2_groups += k.groups; }
            else { t.wave_ms += ms; t.wave_launches++; t.wave_rows += k.rows; t.wave_groups += k.groups; }
            if (ctx->launch_log.size() < 65536) ctx->launch_log.push_back(ef_launch_record{k.which, k.groups, k.rows, ms});
        }
        ctx->timing_pool.push_back(k.e0);
        ctx->timing_pool.push_back(k.e1);
    }
    ctx->kspans.clear();
}

extern "C" int32_t ef_set_kernel_timing(ef_ctx* ctx, int32_t on) {
    EF_CHECK_CTX(ctx);
    ctx->time_kernels = on ? 1 : 0;
    return EF_OK;
}

extern "C" int32_t ef_get_kernel_times(ef_ctx* ctx, ef_kernel_times* out, int32_t reset) {
    EF_CHECK_CTX(ctx);
    if (!out) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_get_kernel_times: null");
    drain_kernel_spans(ctx);
    *out = ctx->ktimes;
    if (reset) ctx->ktimes = ef_kernel_times();
    return EF_OK;
}

extern "C" int32_t ef_get_launch_log(ef_ctx* ctx, ef_launch_record* out, int32_t max_records, int32_t* n_out, int32_t reset) {
    EF_CHECK_CTX(ctx);
    if (!n_out || max_records < 0 || (max_records > 0 && !out)) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_get_launch_log: bad argument");
    drain_kernel_spans(ctx);
    const int32_t n = (int32_t)std::min<size_t>((size_t)max_records, ctx->launch_log.size());
    for (int32_t i = 0; i < n; ++i) out[i] = ctx->launch_log[i];
    *n_out = n;
    if (reset) ctx->launch_log.clear();
    return EF_OK;
}
