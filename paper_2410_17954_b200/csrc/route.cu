// a1: router logits + top-k + gate weights  (Eq. 1-2, L40-46; R1-R3).
//
// logits[T,E] = x[T,d] . Wr[E,d]^T + b is a skinny GEMM (N = E <= 256): HBM-bound on x for E = 8, ALU-bound on
// plain FMA for E = 64 (2*d*E flop per token), so the contraction runs on the legacy tensor path (mma.sync
// m16n8k16, bf16 x bf16 -> fp32) -- the tile is far too small for a tcgen05 pipeline, and the kernel is
// latency-bound, not throughput-bound.
//
// One CTA = 16 tokens (one MMA M tile) x all experts, 8 warps splitting K: warp w takes the 32-wide k chunks
// w, w+8, ...  Fragments come straight from global memory with 128-bit loads: thread (g, t) of a warp loads
// elements [8t, 8t+8) of the chunk from row g (and g+8) of x and from row g of each 8-expert tile of Wr, and
// feeds elements (4s, 4s+1 | 4s+2, 4s+3) to MMA step s = 0, 1.  That is a permutation of k inside the chunk,
// applied identically to both operands, so every product still meets its partner.  Per-warp partial tiles are
// summed across the 8 warps through shared memory in a fixed order (deterministic), the bias is added, and
// each warp then finishes two tokens: k rounds of warp arg-max (ties -> lower expert index) and the gate
// weights with expf in fp32.
#include <cuda_bf16.h>

#include "ef_internal.h"

namespace {

constexpr int kWarps = 8;
constexpr int kTok = 16;          // tokens per CTA
constexpr int kEChunk = 64;       // experts per accumulation pass (8 MMA N tiles)
constexpr int kPartLd = 72;       // padded row stride of the partial tiles (floats)

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// (value, index) argmax with ties -> smaller index
__device__ __forceinline__ void warp_argmax(float& v, int& i) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        float ov = __shfl_xor_sync(0xffffffffu, v, o);
        int oi = __shfl_xor_sync(0xffffffffu, i, o);
        if (ov > v || (ov == v && oi < i)) { v = ov; i = oi; }
    }
}

__device__ __forceinline__ void mma_bf16(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                         uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// kUnroll: k chunks whose x fragments are in flight per warp before the MMAs consume them (the kernel is bound by load
// latency: more independent 128-bit loads per thread, as far as the registers of the 8-expert-tile loop allow)
template <int kUnroll>
__global__ void __launch_bounds__(kWarps * 32)
route_topk_kernel(const uint4* __restrict__ x, const uint4* __restrict__ wr, const float* __restrict__ bias,
                  int64_t bias_stride, int T, int d8, int E, int k, int renorm, int32_t* __restrict__ idx,
                  float* __restrict__ w, float* __restrict__ logits_out) {
    extern __shared__ float smem_f[];
    float* s_part = smem_f;                                   // [kWarps][kTok][kPartLd]
    float* s_logits = smem_f + kWarps * kTok * kPartLd;       // [kTok][E]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, tq = lane & 3;
    const int t0 = blockIdx.x * kTok;
    const int n_chunks = d8 >> 2;                             // 32-element k chunks (d % 64 == 0)
    const uint4 zero4 = make_uint4(0, 0, 0, 0);
    const bool r0_ok = t0 + g < T, r1_ok = t0 + g + 8 < T;
    const uint4* xa = x + (int64_t)(t0 + g) * d8 + tq;
    const uint4* xb = x + (int64_t)(t0 + g + 8) * d8 + tq;

    for (int e0 = 0; e0 < E; e0 += kEChunk) {
        float acc[kEChunk / 8][4];
#pragma unroll
        for (int n = 0; n < kEChunk / 8; ++n) { acc[n][0] = acc[n][1] = acc[n][2] = acc[n][3] = 0.f; }
        const int n_tiles = min(kEChunk / 8, (E - e0 + 7) >> 3);
        for (int c0 = warp; c0 < n_chunks; c0 += kWarps * kUnroll) {
            uint4 a_lo[kUnroll], a_hi[kUnroll];
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                const int c = c0 + u * kWarps;
                a_lo[u] = (r0_ok && c < n_chunks) ? xa[c * 4] : zero4;
                a_hi[u] = (r1_ok && c < n_chunks) ? xb[c * 4] : zero4;
            }
#pragma unroll
            for (int n = 0; n < kEChunk / 8; ++n) {
                if (n < n_tiles) {
                    const int e = e0 + n * 8 + g;
                    uint4 b[kUnroll];
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) {
                        const int c = c0 + u * kWarps;
                        b[u] = (e < E && c < n_chunks) ? __ldg(wr + (int64_t)e * d8 + c * 4 + tq) : zero4;
                    }
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) {
                        mma_bf16(acc[n], a_lo[u].x, a_hi[u].x, a_lo[u].y, a_hi[u].y, b[u].x, b[u].y);
                        mma_bf16(acc[n], a_lo[u].z, a_hi[u].z, a_lo[u].w, a_hi[u].w, b[u].z, b[u].w);
                    }
                }
            }
        }
        // partial tiles -> shared memory, fixed-order sum over the 8 warps, + bias
        float* mine = s_part + warp * kTok * kPartLd;
#pragma unroll
        for (int n = 0; n < kEChunk / 8; ++n) {
            *reinterpret_cast<float2*>(mine + g * kPartLd + n * 8 + 2 * tq) = make_float2(acc[n][0], acc[n][1]);
            *reinterpret_cast<float2*>(mine + (g + 8) * kPartLd + n * 8 + 2 * tq) = make_float2(acc[n][2], acc[n][3]);
        }
        __syncthreads();
        for (int i = threadIdx.x; i < kTok * kEChunk; i += kWarps * 32) {
            const int r = i / kEChunk, col = i % kEChunk;
            if (e0 + col < E) {
                float s = 0.f;
#pragma unroll
                for (int ww = 0; ww < kWarps; ++ww) s += s_part[(ww * kTok + r) * kPartLd + col];
                const int t = t0 + r;
                if (bias && t < T) s += bias[(int64_t)t * bias_stride + e0 + col];
                s_logits[r * E + e0 + col] = s;
            }
        }
        __syncthreads();
    }

    // each warp finishes two tokens
    for (int r = warp; r < kTok; r += kWarps) {
        const int t = t0 + r;
        if (t >= T) break;
        const float* lg = s_logits + r * E;
        if (logits_out)
            for (int e = lane; e < E; e += 32) logits_out[(int64_t)t * E + e] = lg[e];
        // candidates: lane owns experts lane, lane+32, ...  A NaN logit (NaN in x, the router or the bias: undefined input,
        // R2) ranks as -inf, and among equal candidates the lowest untaken index wins, so every pick is a valid expert id
        // whatever the input (an all-NaN row selects experts 0 .. k-1, as the oracle's strict '>' scan does).
        float v[8];
        unsigned taken = 0;                       // bit i: expert lane + 32 i has been picked
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            int e = lane + 32 * i;
            v[i] = (e < E) ? lg[e] : -INFINITY;
            if (v[i] != v[i]) v[i] = -INFINITY;
        }
        float zall = 0.f, m = 0.f, zsel = 0.f, my_val = 0.f;
        int my_idx = 0;
        for (int j = 0; j < k; ++j) {
            float bv = -INFINITY;
            int bi = 0x7fffffff;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                int e = lane + 32 * i;
                if (e < E && !((taken >> i) & 1u) && (v[i] > bv || (v[i] == bv && e < bi))) { bv = v[i]; bi = e; }
            }
            warp_argmax(bv, bi);
            if (j == 0) {
                m = bv;
                if (!renorm) {
                    float z = 0.f;
                    for (int e = lane; e < E; e += 32) z += expf(lg[e] - m);
                    zall = warp_sum(z);
                }
            }
            zsel += expf(bv - m);
            if (lane == j) { my_val = bv; my_idx = bi; }
            if ((bi & 31) == lane) taken |= 1u << (bi >> 5);
        }
        if (lane < k) {
            const float Z = renorm ? zsel : zall;
            idx[(int64_t)t * k + lane] = my_idx;
            w[(int64_t)t * k + lane] = expf(my_val - m) / Z;
        }
    }
}

}  // namespace

int32_t efk_route_topk(ef_ctx* ctx, cudaStream_t st, const void* x, const void* wr, const float* bias,
                       int64_t bias_stride, int T, int renorm, int32_t* idx, float* w, float* logits) {
    if (T == 0) return EF_OK;
    const int E = ctx->cfg.n_experts, d = ctx->cfg.d_model, k = ctx->cfg.top_k;
    dim3 grid((T + kTok - 1) / kTok), block(kWarps * 32);
    const size_t smem = ((size_t)kWarps * kTok * kPartLd + (size_t)kTok * E) * sizeof(float);
    if (smem > 48 * 1024 && !ctx->route_smem_set) {
        EF_CUDA(ctx, cudaFuncSetAttribute(route_topk_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
        EF_CUDA(ctx, cudaFuncSetAttribute(route_topk_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
        ctx->route_smem_set = true;
    }
    if (E <= 16)
        route_topk_kernel<8><<<grid, block, smem, st>>>((const uint4*)x, (const uint4*)wr, bias, bias_stride, T, d / 8, E, k,
                                                        renorm, idx, w, logits);
    else
        route_topk_kernel<4><<<grid, block, smem, st>>>((const uint4*)x, (const uint4*)wr, bias, bias_stride, T, d / 8, E, k,
                                                        renorm, idx, w, logits);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    return EF_OK;
}
