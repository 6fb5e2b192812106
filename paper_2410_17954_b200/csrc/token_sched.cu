// f1: Token Scheduler (§3.3): rebatch 2T tokens into two batches of T by balanced 2-means over
// the Hamming similarity of their routing paths (Eq. 6), so that each batch activates fewer experts (Eq. 5).
// Readings R26-R29 fix what the missing appendix would: cluster 0 = the T tokens with the largest
// margin S[i,c0] - S[i,c1], ties to the lower index; centroid = medoid; converged = centroids unchanged.
//
// Kernels (all on the caller's stream, no host synchronisation -- the iteration loop is unrolled on the host to
// max_iter rounds and a device-side `done` flag turns the rounds after convergence into empty launches):
//   ts_pack_kernel     r[N, LE] bytes -> bit-packed paths P[N, Wd] (ballot), Wd = ceil(LE / 32)
//   ts_hamming_kernel  d_ij = sum_w popc(P[i,w] ^ P[j,w]) -> uint16 D[N, N]; 64 x 64 tiles, 4 x 4 outputs per thread,
//                      word chunks staged in shared memory, tile transposed through shared memory so that every row
//                      segment is written with 16-byte stores.  ALU-bound (xor + popc + add per pair and word).
//   ts_assign_kernel   one CTA: applies the previous round's centroid update, then margins m_i = D[c1,i] - D[c0,i]
//                      (rows of the symmetric D: contiguous), the T-th largest margin by bisection over its integer
//                      range, ties ranked by index with a block scan -> batch_of[N] and a membership bit mask
//   ts_medoid_kernel   one warp per token: sum of D[i, j] over the tokens j of i's cluster (16-byte loads of the row,
//                      mask bits from shared memory), 64-bit atomicMin of (sum << 32 | i) per cluster.  Reads D once
//                      per round: L2/HBM-bound (2 N^2 bytes).
//   ts_finalize_kernel last centroid update, perm (T_1 ascending, then T_2 ascending -- the "Reindex" map of §3.3.1,
//                      P:L151), Eq. 5 objective of the result and of the incoming batching (OR over tokens, R14)
#include <limits.h>

#include "ef_internal.h"

namespace {

constexpr int TS_TILE = 64;       // tokens per Hamming tile side
constexpr int TS_WC = 32;         // path words per shared-memory chunk
constexpr int TS_BLOCK = 1024;    // threads of the single-CTA kernels
constexpr int TS_MAX_PER_THREAD = EF_TS_MAX_TOKENS / TS_BLOCK;

struct TsState {
    int32_t c0, c1;
    int32_t done, converged, iters, max_iter;
    unsigned long long best[2];   // (summed distance << 32 | token) minimum per cluster
};

__global__ void __launch_bounds__(256)
ts_pack_kernel(const uint8_t* __restrict__ r, int N, int LE, int Wd, uint32_t* __restrict__ P) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= N) return;
    const uint8_t* row = r + (size_t)warp * LE;
    for (int w = 0; w < Wd; ++w) {
        const int c = w * 32 + lane;
        const unsigned bits = __ballot_sync(0xffffffffu, c < LE && row[c] != 0);
        if (lane == 0) P[(size_t)warp * Wd + w] = bits;
    }
}

__global__ void __launch_bounds__(256)
ts_hamming_kernel(const uint32_t* __restrict__ P, int N, int Wd, uint16_t* __restrict__ D) {
    __shared__ uint32_t sA[TS_TILE][TS_WC + 1];
    __shared__ uint32_t sB[TS_TILE][TS_WC + 1];
    __shared__ __align__(16) uint16_t sOut[TS_TILE][TS_TILE + 8];
    const int i0 = blockIdx.y * TS_TILE, j0 = blockIdx.x * TS_TILE;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    uint32_t acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0;
    for (int w0 = 0; w0 < Wd; w0 += TS_WC) {
        const int wc = min(TS_WC, Wd - w0);
        for (int t = threadIdx.x; t < TS_TILE * TS_WC; t += 256) {
            const int rr = t / TS_WC, c = t % TS_WC;
            const bool okc = c < wc;
            sA[rr][c] = (okc && i0 + rr < N) ? P[(size_t)(i0 + rr) * Wd + w0 + c] : 0u;
            sB[rr][c] = (okc && j0 + rr < N) ? P[(size_t)(j0 + rr) * Wd + w0 + c] : 0u;
        }
        __syncthreads();
        for (int w = 0; w < wc; ++w) {
            uint32_t a4[4], b4[4];
#pragma unroll
            for (int a = 0; a < 4; ++a) a4[a] = sA[ty + 16 * a][w];
#pragma unroll
            for (int b = 0; b < 4; ++b) b4[b] = sB[tx + 16 * b][w];
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) acc[a][b] += __popc(a4[a] ^ b4[b]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) sOut[ty + 16 * a][tx + 16 * b] = (uint16_t)acc[a][b];
    __syncthreads();
    // 64 rows x 128 bytes: 8 threads per row, 16 bytes each (N is even, rows of D are 2N bytes: 16-byte alignment of a
    // segment needs j0 * 2 % 16 == 0, true, and N * 2 % 16 == 0, i.e. N % 8 == 0 -- otherwise fall back to 2-byte stores)
    const bool vec = (N & 7) == 0;
    for (int t = threadIdx.x; t < TS_TILE * 8; t += 256) {
        const int rr = t >> 3, c8 = (t & 7) * 8;
        if (i0 + rr >= N) continue;
        uint16_t* dst = D + (size_t)(i0 + rr) * N + j0 + c8;
        if (vec && j0 + c8 + 8 <= N) {
            *reinterpret_cast<uint4*>(dst) = *reinterpret_cast<const uint4*>(&sOut[rr][c8]);
        } else {
            for (int q = 0; q < 8 && j0 + c8 + q < N; ++q) dst[q] = sOut[rr][c8 + q];
        }
    }
}

// previous round's update: n = argmin per cluster; unchanged -> converged (R28), else the centroids move
__device__ __forceinline__ void ts_apply_update(TsState* st) {
    const int n0 = (int)(st->best[0] & 0xffffffffull), n1 = (int)(st->best[1] & 0xffffffffull);
    if (n0 == st->c0 && n1 == st->c1) { st->done = 1; st->converged = 1; }
    else { st->c0 = n0; st->c1 = n1; }
}

__device__ __forceinline__ int block_sum(int v, int* s_red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) s_red[warp] = v;
    __syncthreads();
    int t = (lane < TS_BLOCK / 32) ? s_red[lane] : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    return t;
}

// exclusive rank of this thread's flag among the flags of the block (thread order), plus the block total
__device__ __forceinline__ int block_rank(bool flag, int* s_warp, int* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned m = __ballot_sync(0xffffffffu, flag);
    __syncthreads();
    if (lane == 0) s_warp[warp] = __popc(m);
    __syncthreads();
    int before = 0, all = 0;
    for (int w = 0; w < TS_BLOCK / 32; ++w) {
        const int c = s_warp[w];
        if (w < warp) before += c;
        all += c;
    }
    *total = all;
    return before + __popc(m & ((1u << lane) - 1u));
}

__global__ void __launch_bounds__(TS_BLOCK)
ts_assign_kernel(const uint16_t* __restrict__ D, int N, int LE, int round, TsState* st, int32_t* __restrict__ batch_of,
                 uint32_t* __restrict__ member_bits) {
    __shared__ int s_red[TS_BLOCK / 32];
    __shared__ int s_c[3];
    if (threadIdx.x == 0) {
        if (round > 0 && !st->done) ts_apply_update(st);
        if (!st->done && round >= st->max_iter) st->done = 1;
        if (!st->done) {
            st->iters = round + 1;
            st->best[0] = ~0ull;
            st->best[1] = ~0ull;
        }
        s_c[0] = st->c0; s_c[1] = st->c1; s_c[2] = st->done;
    }
    __syncthreads();
    if (s_c[2]) return;
    const int c0 = s_c[0], c1 = s_c[1], T = N >> 1;
    const uint16_t* r0 = D + (size_t)c0 * N;
    const uint16_t* r1 = D + (size_t)c1 * N;
    int m[TS_MAX_PER_THREAD];
#pragma unroll
    for (int q = 0; q < TS_MAX_PER_THREAD; ++q) {
        const int i = q * TS_BLOCK + threadIdx.x;
        m[q] = (i < N) ? (int)r1[i] - (int)r0[i] : INT_MIN;
    }
    // largest threshold th with #{m_i >= th} >= T (bisection over [-LE, LE]; #{m_i >= -LE} = N >= T)
    int lo = -LE, hi = LE + 1;
    while (hi - lo > 1) {
        const int mid = lo + ((hi - lo) >> 1);
        int c = 0;
#pragma unroll
        for (int q = 0; q < TS_MAX_PER_THREAD; ++q) c += (m[q] >= mid) ? 1 : 0;
        c = block_sum(c, s_red);
        if (c >= T) lo = mid; else hi = mid;
    }
    const int th = lo;
    int above = 0;
#pragma unroll
    for (int q = 0; q < TS_MAX_PER_THREAD; ++q) above += (m[q] > th) ? 1 : 0;
    above = block_sum(above, s_red);
    const int quota = T - above;          // ties admitted to cluster 0, in index order (R27)
    int base = 0;
#pragma unroll
    for (int q = 0; q < TS_MAX_PER_THREAD; ++q) {
        if (q * TS_BLOCK >= N) break;      // uniform
        const int i = q * TS_BLOCK + threadIdx.x;
        const bool tie = (i < N) && m[q] == th;
        int total;
        const int rank = base + block_rank(tie, s_red, &total);
        base += total;
        const bool in0 = (i < N) && (m[q] > th || (tie && rank < quota));
        const unsigned bits = __ballot_sync(0xffffffffu, in0);
        if (i < N) batch_of[i] = in0 ? 0 : 1;
        if ((threadIdx.x & 31) == 0 && q * TS_BLOCK + (int)threadIdx.x < N) member_bits[i >> 5] = bits;
    }
}

constexpr int TS_ROWS_PER_CTA = 32;

__global__ void __launch_bounds__(256)
ts_medoid_kernel(const uint16_t* __restrict__ D, int N, const int32_t* __restrict__ batch_of,
                 const uint32_t* __restrict__ member_bits, TsState* st) {
    extern __shared__ uint32_t s_bits[];      // [ceil(N / 32)] bit j set <=> token j is in cluster 0
    if (st->done) return;
    const int nw = (N + 31) >> 5;
    for (int t = threadIdx.x; t < nw; t += blockDim.x) s_bits[t] = member_bits[t];
    __syncthreads();
    const uint8_t* s_bytes = reinterpret_cast<const uint8_t*>(s_bits);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool vec = (N & 7) == 0;
    for (int rr = warp; rr < TS_ROWS_PER_CTA; rr += 8) {
        const int i = blockIdx.x * TS_ROWS_PER_CTA + rr;
        if (i >= N) break;
        const uint16_t* row = D + (size_t)i * N;
        uint32_t s_all = 0, s_0 = 0;
        if (vec) {
            for (int j = lane * 8; j < N; j += 256) {
                const uint4 v = *reinterpret_cast<const uint4*>(row + j);
                const uint32_t mb = s_bytes[j >> 3];
                const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t a = w[q] & 0xffffu, b = w[q] >> 16;
                    s_all += a + b;
                    s_0 += ((mb >> (2 * q)) & 1u) * a + ((mb >> (2 * q + 1)) & 1u) * b;
                }
            }
        } else {
            for (int j = lane; j < N; j += 32) {
                const uint32_t a = row[j];
                s_all += a;
                s_0 += ((s_bits[j >> 5] >> (j & 31)) & 1u) * a;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            s_all += __shfl_xor_sync(0xffffffffu, s_all, o);
            s_0 += __shfl_xor_sync(0xffffffffu, s_0, o);
        }
        if (lane == 0) {
            const int b = batch_of[i];
            const unsigned long long sum = b ? (s_all - s_0) : s_0;
            atomicMin(&st->best[b], (sum << 32) | (unsigned long long)(uint32_t)i);
        }
    }
}

__global__ void __launch_bounds__(TS_BLOCK)
ts_finalize_kernel(const uint32_t* __restrict__ P, int N, int LE, int Wd, TsState* st, const int32_t* __restrict__ batch_of,
                   int32_t* __restrict__ perm, int32_t* __restrict__ info, uint8_t* __restrict__ batch_paths) {
    extern __shared__ uint32_t s_or[];        // [4][Wd]: new batch 0, new batch 1, incoming batch 0, incoming batch 1
    __shared__ int s_red[TS_BLOCK / 32];
    if (threadIdx.x == 0 && !st->done) { ts_apply_update(st); st->done = 1; }
    for (int t = threadIdx.x; t < 4 * Wd; t += TS_BLOCK) s_or[t] = 0;
    __syncthreads();
    const int T = N >> 1;
    // perm: members of cluster 0 in ascending index, then members of cluster 1 (each cluster holds exactly T tokens)
    int base0 = 0;
    for (int q = 0; q * TS_BLOCK < N; ++q) {
        const int i = q * TS_BLOCK + threadIdx.x;
        const bool in0 = (i < N) && batch_of[i] == 0;
        int total;
        const int r0 = base0 + block_rank(in0, s_red, &total);
        base0 += total;
        if (i < N) perm[in0 ? r0 : T + (i - r0)] = i;
    }
    // Eq. 5 with OR (R14)
    for (int t = threadIdx.x; t < N * Wd; t += TS_BLOCK) {
        const int i = t / Wd, w = t - i * Wd;
        const uint32_t v = P[t];
        if (v) {
            atomicOr(&s_or[batch_of[i] * Wd + w], v);
            atomicOr(&s_or[(2 + (i >= T ? 1 : 0)) * Wd + w], v);
        }
    }
    __syncthreads();
    if (batch_paths)
        for (int t = threadIdx.x; t < 2 * LE; t += TS_BLOCK) {
            const int b = t / LE, c = t - b * LE;
            batch_paths[t] = (uint8_t)((s_or[b * Wd + (c >> 5)] >> (c & 31)) & 1u);
        }
    int after = 0, before = 0;
    for (int t = threadIdx.x; t < 2 * Wd; t += TS_BLOCK) {
        after += __popc(s_or[t]);
        before += __popc(s_or[2 * Wd + t]);
    }
    after = block_sum(after, s_red);
    before = block_sum(before, s_red);
    if (threadIdx.x == 0) {
        info[0] = st->iters; info[1] = st->converged; info[2] = st->c0; info[3] = st->c1;
        info[4] = after; info[5] = before; info[6] = 0; info[7] = 0;
    }
}

// ---- decode-sized problems (N <= 256): the whole schedule in ONE CTA, distance matrix in shared memory ------------
// Same arithmetic as the multi-kernel path (same margins, same tie rules), but one launch instead of 3 + 2 * max_iter:
// at N = 2 x 16 .. 2 x 64 decode tokens the multi-kernel path is all launch latency.
constexpr int TS_SMALL_N = 256;

__global__ void __launch_bounds__(TS_BLOCK)
ts_small_kernel(const uint8_t* __restrict__ r, int N, int LE, int Wd, int c0, int c1, int max_iter,
                int32_t* __restrict__ batch_of, int32_t* __restrict__ perm, int32_t* __restrict__ info,
                uint8_t* __restrict__ batch_paths) {
    extern __shared__ __align__(16) uint8_t ts_smem[];
    const int ldp = Wd | 1;                                   // odd word stride: conflict-free column walks
    const int ldd = N + 2;
    uint32_t* sP = reinterpret_cast<uint32_t*>(ts_smem);      // [N][ldp]
    uint32_t* sOr = sP + (size_t)N * ldp;                     // [4][Wd]
    int* sM = reinterpret_cast<int*>(sOr + 4 * Wd);           // [N] margins
    int* sB = sM + N;                                         // [N] batch_of
    uint16_t* sD = reinterpret_cast<uint16_t*>(sB + N);       // [N][ldd]
    __shared__ unsigned long long s_best[2];
    __shared__ int s_st[5];                                   // c0, c1, done, converged, iters
    __shared__ int s_red[TS_BLOCK / 32];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, T = N >> 1;

    for (int i = warp; i < N; i += TS_BLOCK / 32) {
        const uint8_t* row = r + (size_t)i * LE;
        for (int w = 0; w < Wd; ++w) {
            const int c = w * 32 + lane;
            const unsigned bits = __ballot_sync(0xffffffffu, c < LE && row[c] != 0);
            if (lane == 0) sP[i * ldp + w] = bits;
        }
    }
    if (tid == 0) { s_st[0] = c0; s_st[1] = c1; s_st[2] = 0; s_st[3] = 0; s_st[4] = 0; }
    __syncthreads();
    for (int t = tid; t < N * N; t += TS_BLOCK) {
        const int i = t / N, j = t - i * N;
        uint32_t d = 0;
        for (int w = 0; w < Wd; ++w) d += __popc(sP[i * ldp + w] ^ sP[j * ldp + w]);
        sD[i * ldd + j] = (uint16_t)d;
    }
    __syncthreads();

    for (int round = 0; round < max_iter; ++round) {
        const int a0 = s_st[0], a1 = s_st[1];
        if (tid < N) sM[tid] = (int)sD[a1 * ldd + tid] - (int)sD[a0 * ldd + tid];
        if (tid == 0) { s_best[0] = ~0ull; s_best[1] = ~0ull; s_st[4] = round + 1; }
        __syncthreads();
        if (tid < N) {
            // rank in the order (margin descending, index ascending): cluster 0 = ranks [0, T)   (R26, R27)
            const int mi = sM[tid];
            int rank = 0;
            for (int j = 0; j < N; ++j) {
                const int mj = sM[j];
                rank += (mj > mi || (mj == mi && j < tid)) ? 1 : 0;
            }
            sB[tid] = rank < T ? 0 : 1;
        }
        __syncthreads();
        if (tid < N) {
            const int b = sB[tid];
            uint32_t sum = 0;
            for (int j = 0; j < N; ++j) sum += (sB[j] == b) ? (uint32_t)sD[j * ldd + tid] : 0u;   // D is symmetric
            atomicMin(&s_best[b], ((unsigned long long)sum << 32) | (unsigned long long)(uint32_t)tid);
        }
        __syncthreads();
        if (tid == 0) {
            const int n0 = (int)(s_best[0] & 0xffffffffull), n1 = (int)(s_best[1] & 0xffffffffull);
            if (n0 == s_st[0] && n1 == s_st[1]) { s_st[2] = 1; s_st[3] = 1; }
            else { s_st[0] = n0; s_st[1] = n1; }
        }
        __syncthreads();
        if (s_st[2]) break;
    }

    for (int t = tid; t < 4 * Wd; t += TS_BLOCK) sOr[t] = 0;
    __syncthreads();
    if (tid < N) {
        const int b = sB[tid];
        int r0 = 0;
        for (int j = 0; j < tid; ++j) r0 += (sB[j] == 0) ? 1 : 0;
        batch_of[tid] = b;
        perm[b == 0 ? r0 : T + (tid - r0)] = tid;
    }
    for (int t = tid; t < N * Wd; t += TS_BLOCK) {
        const int i = t / Wd, w = t - i * Wd;
        const uint32_t v = sP[i * ldp + w];
        if (v) {
            atomicOr(&sOr[sB[i] * Wd + w], v);
            atomicOr(&sOr[(2 + (i >= T ? 1 : 0)) * Wd + w], v);
        }
    }
    __syncthreads();
    if (batch_paths)
        for (int t = tid; t < 2 * LE; t += TS_BLOCK) {
            const int b = t / LE, c = t - b * LE;
            batch_paths[t] = (uint8_t)((sOr[b * Wd + (c >> 5)] >> (c & 31)) & 1u);
        }
    int after = 0, before = 0;
    for (int t = tid; t < 2 * Wd; t += TS_BLOCK) {
        after += __popc(sOr[t]);
        before += __popc(sOr[2 * Wd + t]);
    }
    after = block_sum(after, s_red);
    before = block_sum(before, s_red);
    if (tid == 0) {
        info[0] = s_st[4]; info[1] = s_st[3]; info[2] = s_st[0]; info[3] = s_st[1];
        info[4] = after; info[5] = before; info[6] = 0; info[7] = 0;
    }
}

size_t ts_small_smem(int N, int Wd) {
    return (size_t)N * (Wd | 1) * 4 + (size_t)4 * Wd * 4 + (size_t)2 * N * 4 + (size_t)N * (N + 2) * 2;
}

__global__ void ts_init_kernel(TsState* st, int c0, int c1, int max_iter) {
    st->c0 = c0; st->c1 = c1; st->done = 0; st->converged = 0; st->iters = 0; st->max_iter = max_iter;
    st->best[0] = ~0ull; st->best[1] = ~0ull;
}

int32_t ts_reserve(ef_ctx* ctx, int N, int Wd, bool need_dist) {
    const size_t packed = (size_t)N * Wd * sizeof(uint32_t), bits = (size_t)((N + 31) / 32) * sizeof(uint32_t);
    const size_t dist = need_dist ? (size_t)N * N * sizeof(uint16_t) : 0;
    if (!ctx->ts_state) EF_CUDA(ctx, cudaMalloc(&ctx->ts_state, sizeof(TsState)));
    if (packed + bits > ctx->ts_small_bytes) {
        if (ctx->ts_small) EF_CUDA(ctx, cudaFree(ctx->ts_small));
        ctx->ts_small = nullptr; ctx->ts_small_bytes = 0;
        if (cudaMalloc(&ctx->ts_small, packed + bits) != cudaSuccess) { cudaGetLastError(); return ef_fail(ctx, EF_ERR_OOM, "token scheduler workspace"); }
        ctx->ts_small_bytes = packed + bits;
    }
    if (dist > ctx->ts_dist_bytes) {
        if (ctx->ts_dist) EF_CUDA(ctx, cudaFree(ctx->ts_dist));
        ctx->ts_dist = nullptr; ctx->ts_dist_bytes = 0;
        if (cudaMalloc(&ctx->ts_dist, dist) != cudaSuccess) { cudaGetLastError(); return ef_fail(ctx, EF_ERR_OOM, "token scheduler distance matrix"); }
        ctx->ts_dist_bytes = dist;
    }
    return EF_OK;
}

int32_t ts_distances(ef_ctx* ctx, cudaStream_t st, const uint8_t* paths, int N, int LE, uint16_t* D) {
    const int Wd = (LE + 31) / 32;
    uint32_t* P = (uint32_t*)ctx->ts_small;
    ts_pack_kernel<<<(N * 32 + 255) / 256, 256, 0, st>>>(paths, N, LE, Wd, P);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    const int nt = (N + TS_TILE - 1) / TS_TILE;
    ts_hamming_kernel<<<dim3(nt, nt), 256, 0, st>>>(P, N, Wd, D);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    return EF_OK;
}

}  // namespace

// ---- the no-allocation entry point (ef.h: ef_path_hamming_static) ------------------------------------------------------
// Scratch for the bit-packed paths of ONE call, in the library's image instead of in cudaMalloc'ed memory:
// EF_STATIC_SCRATCH_BYTES (1 MiB) on every GPU that loads the library, until the process exits.  In HOST code the name
// below is a host-side stand-in, not a device address; the address is resolved once per device, at set-up (ef_create, with
// the ctx's device current), by cudaGetSymbolAddress, and that pointer is what the kernels are given.
static __device__ __align__(256) uint32_t g_ts_static_scratch[EF_STATIC_SCRATCH_BYTES / sizeof(uint32_t)];

// set-up: called by ef_create with the ctx's device current.  A failure is remembered, not fatal: only
// ef_path_hamming_static needs the address, and it reports the failure when it is called.
void efk_token_sched_static_init(ef_ctx* ctx) {
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_ts_static_scratch);
    if (e != cudaSuccess) {
        cudaGetLastError();
        ptr = nullptr;
    }
    ctx->ts_static_scratch = ptr;
    ctx->ts_static_err = (int32_t)e;
}

// No cudaMalloc, cudaFree or allocating library routine on this path: two kernel launches on the caller's stream.
// Nothing in the scratch has to start at zero: ts_pack_kernel overwrites every word ts_hamming_kernel reads (rows < N,
// words < Wd), so the previous call's contents are never seen.
int32_t efk_path_hamming_static(ef_ctx* ctx, cudaStream_t st, const uint8_t* paths, int N, int LE, uint16_t* dist_out) {
    const int Wd = (LE + 31) / 32;
    const size_t need = (size_t)N * Wd * sizeof(uint32_t);
    if (need > (size_t)EF_STATIC_SCRATCH_BYTES)
        return ef_fail(ctx, EF_ERR_CAPACITY, "ef_path_hamming_static: N * ceil(LE / 32) * 4 = %zu bytes of packed paths exceed the static "
                       "scratch of %d bytes (use ef_path_hamming, which allocates)", need, (int)EF_STATIC_SCRATCH_BYTES);
    if (!ctx->ts_static_scratch)
        return ef_fail(ctx, EF_ERR_CUDA, "ef_path_hamming_static: cudaGetSymbolAddress of the static scratch failed at ef_create: %s",
                       cudaGetErrorString((cudaError_t)ctx->ts_static_err));
    uint32_t* P = (uint32_t*)ctx->ts_static_scratch;
    ts_pack_kernel<<<(N * 32 + 255) / 256, 256, 0, st>>>(paths, N, LE, Wd, P);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    const int nt = (N + TS_TILE - 1) / TS_TILE;
    ts_hamming_kernel<<<dim3(nt, nt), 256, 0, st>>>(P, N, Wd, dist_out);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    return EF_OK;
}

void efk_token_sched_free(ef_ctx* ctx) {
    if (ctx->ts_state) cudaFree(ctx->ts_state);
    if (ctx->ts_small) cudaFree(ctx->ts_small);
    if (ctx->ts_dist) cudaFree(ctx->ts_dist);
    ctx->ts_state = nullptr; ctx->ts_small = nullptr; ctx->ts_dist = nullptr;
}

int32_t efk_path_hamming(ef_ctx* ctx, cudaStream_t st, const uint8_t* paths, int N, int LE, uint16_t* dist_out) {
    int32_t rc = ts_reserve(ctx, N, (LE + 31) / 32, false);
    if (rc != EF_OK) return rc;
    return ts_distances(ctx, st, paths, N, LE, dist_out);
}

int32_t efk_token_schedule(ef_ctx* ctx, cudaStream_t st, const uint8_t* paths, int N, int LE, int c0, int c1,
                           int max_iter, int32_t* batch_of, int32_t* perm, int32_t* info, uint8_t* batch_paths) {
    const int Wd = (LE + 31) / 32;
    if (N <= TS_SMALL_N && ts_small_smem(N, Wd) <= 200 * 1024 && !ctx->ts_force_multi) {
        const size_t smem = ts_small_smem(N, Wd);
        if (!ctx->ts_small_attr) {
            EF_CUDA(ctx, cudaFuncSetAttribute(ts_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
            ctx->ts_small_attr = true;
        }
        ts_small_kernel<<<1, TS_BLOCK, smem, st>>>(paths, N, LE, Wd, c0, c1, max_iter, batch_of, perm, info, batch_paths);
        ctx->launches++;
        EF_CUDA(ctx, cudaGetLastError());
        return EF_OK;
    }
    int32_t rc = ts_reserve(ctx, N, Wd, true);
    if (rc != EF_OK) return rc;
    uint16_t* D = (uint16_t*)ctx->ts_dist;
    uint32_t* P = (uint32_t*)ctx->ts_small;
    uint32_t* bits = P + (size_t)N * Wd;
    TsState* state = (TsState*)ctx->ts_state;
    ts_init_kernel<<<1, 1, 0, st>>>(state, c0, c1, max_iter);
    ctx->launches++;
    rc = ts_distances(ctx, st, paths, N, LE, D);
    if (rc != EF_OK) return rc;
    const size_t bits_smem = (size_t)((N + 31) / 32) * sizeof(uint32_t);
    for (int round = 0; round < max_iter; ++round) {
        ts_assign_kernel<<<1, TS_BLOCK, 0, st>>>(D, N, LE, round, state, batch_of, bits);
        ts_medoid_kernel<<<(N + TS_ROWS_PER_CTA - 1) / TS_ROWS_PER_CTA, 256, bits_smem, st>>>(D, N, batch_of, bits, state);
        ctx->launches += 2;
    }
    ts_finalize_kernel<<<1, TS_BLOCK, (size_t)4 * Wd * sizeof(uint32_t), st>>>(P, N, LE, Wd, state, batch_of, perm, info, batch_paths);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    return EF_OK;
}
