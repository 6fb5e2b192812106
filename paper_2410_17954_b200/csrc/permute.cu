// a2: permute tokens by expert (dispatch implied by PAPER.md L21, L68; R5).
//
// Two launches.
//  (1) permute_index_kernel -- one thread-block cluster (1 CTA per ~1024 pairs, at most 8) of 32 warps each.  Stable
//      counting sort of the R = T*k flat pairs: each warp of each CTA owns a contiguous chunk of pairs (chunk order =
//      pair order); the CTAs exchange their per-expert totals through distributed shared memory; per-warp histograms
//      (__match_any_sync groups equal keys, one lane adds the group size: no atomics), a scan over
//      warps then over experts, then every pair's row = offsets[e] + (pairs of e in earlier warps)
//      + (rank inside the warp's running chunk).  Also mirrors counts into pinned host memory.
//  (2) gather_rows_kernel -- HBM-bound row copy x[src[row]/k,:] -> x_perm[row,:], one warp per row,
//      128-bit loads/stores (reads 2*d bytes per token once from HBM -- the k re-reads hit L2 --
//      and writes 2*d*k bytes per token).
#include <algorithm>

#include "ef_internal.h"

namespace {

constexpr int kIdxWarps = 32;
constexpr int kBatch = 8;          // key loads in flight per lane

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// read an int32 at the same shared-memory offset in CTA `rank` of the cluster (distributed shared memory)
__device__ __forceinline__ int32_t ld_dsmem(const int32_t* p, uint32_t rank) {
    uint32_t a = (uint32_t)__cvta_generic_to_shared(p), ra;
    int32_t v;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(a), "r"(rank));
    asm volatile("ld.shared::cluster.s32 %0, [%1];" : "=r"(v) : "r"(ra) : "memory");
    return v;
}

// One thread-block CLUSTER of C CTAs (C = 1 for decode-sized problems, up to 8): CTA c, warp w owns the contiguous
// chunk number c * 32 + w of the pairs, so chunk order = pair order and the sort stays stable.
__global__ void __launch_bounds__(kIdxWarps * 32)
permute_index_kernel(const int32_t* __restrict__ idx, int R, int E, int32_t* __restrict__ counts,
                     int32_t* __restrict__ offsets, int32_t* __restrict__ src, int32_t* __restrict__ inv,
                     int32_t* counts_host, int32_t* err_host) {
    extern __shared__ int32_t sm[];
    int32_t* hist = sm;                       // [kIdxWarps][E]
    int32_t* s_off = sm + kIdxWarps * E;      // [E + 1]
    int32_t* s_tot = s_off + E + 1;           // [E]: pairs of expert e in this CTA (read by the peers)
    int32_t* s_base = s_tot + E;              // [E]: pairs of expert e in earlier CTAs of the cluster
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t crank = cluster_ctarank(), csize = cluster_nctarank();
    for (int i = threadIdx.x; i < kIdxWarps * E; i += blockDim.x) hist[i] = 0;
    __syncthreads();

    // contiguous chunk per warp, multiple of 32 so that iterations are lane-aligned
    int chunk = (R + kIdxWarps * (int)csize - 1) / (kIdxWarps * (int)csize);
    chunk = (chunk + 31) & ~31;
    const int lo = min(R, ((int)crank * kIdxWarps + warp) * chunk), hi = min(R, lo + chunk);
    int32_t* myh = hist + warp * E;

    // keys are fetched kBatch iterations ahead (independent loads in flight)
    for (int base0 = lo; base0 < hi; base0 += 32 * kBatch) {
        int keys[kBatch];
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            const int p = base0 + u * 32 + lane;
            keys[u] = (p < hi) ? idx[p] : (E + lane);    // invalid lanes get unique keys
        }
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            if (base0 + u * 32 >= hi) break;
            // a key outside [0, E) (caller-supplied top-k indices are not trusted) is routed nowhere: it gets a lane-unique
            // key like the lanes past the end, is left out of every count, and raises the error word the host checks
            const bool in_range = (unsigned)keys[u] < (unsigned)E;
            const bool valid = base0 + u * 32 + lane < hi && in_range;
            const int key = in_range ? keys[u] : (E + lane);
            const unsigned mask = __match_any_sync(0xffffffffu, key);
            if (valid && lane == (__ffs(mask) - 1)) myh[key] += __popc(mask);
            __syncwarp();
        }
    }
    __syncthreads();

    // scan over this CTA's warps for each expert: hist[w][e] becomes the number of e-pairs in warps < w
    for (int e = threadIdx.x; e < E; e += blockDim.x) {
        int run = 0;
        for (int w = 0; w < kIdxWarps; ++w) {
            int c = hist[w * E + e];
            hist[w * E + e] = run;
            run += c;
        }
        s_tot[e] = run;
    }
    cluster_sync();                           // every CTA's totals are visible to its peers
    for (int e = threadIdx.x; e < E; e += blockDim.x) {
        int before = 0, all = 0;
        for (uint32_t c = 0; c < csize; ++c) {
            const int v = (c == crank) ? s_tot[e] : ld_dsmem(s_tot + e, c);
            if (c < crank) before += v;
            all += v;
        }
        s_base[e] = before;
        s_off[e + 1] = all;   // temporarily: counts, shifted by one
        if (crank == 0) {
            counts[e] = all;
            if (counts_host) counts_host[e] = all;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        // E <= 256: a serial scan by one thread costs well under a microsecond
        s_off[0] = 0;
        for (int e = 0; e < E; ++e) s_off[e + 1] += s_off[e];
    }
    __syncthreads();
    if (crank == 0) {
        for (int e = threadIdx.x; e <= E; e += blockDim.x) offsets[e] = s_off[e];
    }

    for (int base0 = lo; base0 < hi; base0 += 32 * kBatch) {
        int keys[kBatch];
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            const int p = base0 + u * 32 + lane;
            keys[u] = (p < hi) ? idx[p] : (E + lane);
        }
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            if (base0 + u * 32 >= hi) break;
            const int p = base0 + u * 32 + lane;
            const bool in_range = (unsigned)keys[u] < (unsigned)E;
            const bool valid = p < hi && in_range;
            const int key = in_range ? keys[u] : (E + lane);
            const unsigned mask = __match_any_sync(0xffffffffu, key);
            const int rank = __popc(mask & ((1u << lane) - 1u));
            if (valid) {
                const int row = s_off[key] + s_base[key] + myh[key] + rank;
                inv[p] = row;
                src[row] = p;
            } else if (p < hi) {
                inv[p] = -1;                      // ef_combine skips it
                if (err_host) *err_host = 1;
            }
            __syncwarp();
            if (valid && lane == (__ffs(mask) - 1)) myh[key] += __popc(mask);
            __syncwarp();
        }
    }
    if (counts_host || err_host) __threadfence_system();
    cluster_sync();                           // no CTA exits while a peer may still read its totals
}

__global__ void __launch_bounds__(256)
gather_rows_kernel(const uint4* __restrict__ x, const int32_t* __restrict__ src, int R, int k, int d8,
                   uint4* __restrict__ x_perm, const int32_t* __restrict__ n_rows_dev) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= R) return;
    if (n_rows_dev && warp >= *n_rows_dev) return;     // dispatch: rows past offsets[E] exist only if pairs were skipped
    const int t = src[warp] / k;
    const uint4* in = x + (int64_t)t * d8;
    uint4* out = x_perm + (int64_t)warp * d8;
    int c = lane;
    for (; c + 96 < d8; c += 128) {   // 4 independent 128-bit loads in flight per lane
        uint4 a = in[c], b = in[c + 32], e = in[c + 64], f = in[c + 96];
        out[c] = a; out[c + 32] = b; out[c + 64] = e; out[c + 96] = f;
    }
    for (; c < d8; c += 32) out[c] = in[c];
}

}  // namespace

int32_t efk_permute(ef_ctx* ctx, cudaStream_t st, const int32_t* idx, const void* x, int T, void* x_perm,
                    int32_t* counts, int32_t* offsets, int32_t* src, int32_t* inv, int32_t* counts_host, int32_t* err_host) {
    const int E = ctx->cfg.n_experts, k = ctx->cfg.top_k, d = ctx->cfg.d_model;
    const int R = T * k;
    size_t smem = ((size_t)kIdxWarps * E + 3 * (size_t)E + 1) * sizeof(int32_t);
    // one cluster: a CTA per ~1024 pairs (one 32-pair step per warp), at most 8 (the portable cluster size)
    const int n_cta = std::max(1, std::min(8, (R + 1023) / 1024));
    if (n_cta == 1) {     // a launch without cluster dimensions is a cluster of one CTA
        permute_index_kernel<<<1, kIdxWarps * 32, smem, st>>>(idx, R, E, counts, offsets, src, inv, counts_host, err_host);
        EF_CUDA(ctx, cudaGetLastError());
    } else {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(n_cta);
    cfg.blockDim = dim3(kIdxWarps * 32);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = n_cta; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    EF_CUDA(ctx, cudaLaunchKernelEx(&cfg, permute_index_kernel, idx, R, E, counts, offsets, src, inv, counts_host, err_host));
    }
    ctx->launches++;
    if (R > 0) {
        int blocks = (R * 32 + 255) / 256;
        gather_rows_kernel<<<blocks, 256, 0, st>>>((const uint4*)x, src, R, k, d / 8, (uint4*)x_perm, offsets + E);
        ctx->launches++;
        EF_CUDA(ctx, cudaGetLastError());
    }
    return EF_OK;
}

// "Reindex" of the Token Scheduler (PAPER.md 3.3.1): dst row i = src row perm[i]; the same HBM-bound row copy
// as the dispatch gather, with one source row per destination row.
int32_t efk_reindex_rows(ef_ctx* ctx, cudaStream_t st, const void* src, const int32_t* perm, int n_rows, int64_t row_bytes,
                         void* dst) {
    if (n_rows == 0) return EF_OK;
    const int blocks = (n_rows * 32 + 255) / 256;
    gather_rows_kernel<<<blocks, 256, 0, st>>>((const uint4*)src, perm, n_rows, 1, (int)(row_bytes / 16), (uint4*)dst, nullptr);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    return EF_OK;
}
