// a1: router logits + top-k + gate weights  (Eq. 1-2, L40-46; R1-R3).
//
// HBM-bound: reads x once (2*d bytes per token); Wr (E*d*2 bytes) stays in L1/L2.  One warp per
// token, 128-bit loads, fp32 accumulate, warp-shuffle reductions; top-k by k rounds of warp argmax
// (ties -> lower expert index), gate weights with expf in fp32.
#include <cuda_bf16.h>

#include "ef_internal.h"

namespace {

constexpr int kWarps = 4;
constexpr int kEGroup = 8;

__device__ __forceinline__ float bf_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

__device__ __forceinline__ float dot8(const uint4& a, const uint4& b, float acc) {
    acc = fmaf(bf_lo(a.x), bf_lo(b.x), acc);
    acc = fmaf(bf_hi(a.x), bf_hi(b.x), acc);
    acc = fmaf(bf_lo(a.y), bf_lo(b.y), acc);
    acc = fmaf(bf_hi(a.y), bf_hi(b.y), acc);
    acc = fmaf(bf_lo(a.z), bf_lo(b.z), acc);
    acc = fmaf(bf_hi(a.z), bf_hi(b.z), acc);
    acc = fmaf(bf_lo(a.w), bf_lo(b.w), acc);
    acc = fmaf(bf_hi(a.w), bf_hi(b.w), acc);
    return acc;
}

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

__global__ void __launch_bounds__(kWarps * 32)
route_topk_kernel(const uint4* __restrict__ x, const uint4* __restrict__ wr, const float* __restrict__ bias,
                  int64_t bias_stride, int T, int d8, int E, int k, int renorm, int32_t* __restrict__ idx,
                  float* __restrict__ w, float* __restrict__ logits_out) {
    extern __shared__ float s_logits[];   // [kWarps][E]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int t = blockIdx.x * kWarps + warp;
    if (t >= T) return;
    float* lg = s_logits + warp * E;
    const uint4* xr = x + (int64_t)t * d8;

    for (int e0 = 0; e0 < E; e0 += kEGroup) {
        float acc[kEGroup];
#pragma unroll
        for (int j = 0; j < kEGroup; ++j) acc[j] = 0.f;
        for (int c = lane; c < d8; c += 32) {
            const uint4 xv = xr[c];
#pragma unroll
            for (int j = 0; j < kEGroup; ++j) {
                if (e0 + j < E) {
                    const uint4 wv = __ldg(wr + (int64_t)(e0 + j) * d8 + c);
                    acc[j] = dot8(xv, wv, acc[j]);
                }
            }
        }
#pragma unroll
        for (int j = 0; j < kEGroup; ++j) {
            float s = warp_sum(acc[j]);
            if (lane == 0 && e0 + j < E) {
                float b = bias ? bias[(int64_t)t * bias_stride + e0 + j] : 0.f;
                lg[e0 + j] = s + b;
            }
        }
    }
    __syncwarp();
    if (logits_out)
        for (int e = lane; e < E; e += 32) logits_out[(int64_t)t * E + e] = lg[e];

    // candidates: lane owns experts lane, lane+32, ...
    float v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = lane + 32 * i;
        v[i] = (e < E) ? lg[e] : -INFINITY;
    }
    float zall = 0.f, m = 0.f, zsel = 0.f, my_val = 0.f;
    int my_idx = 0;
    for (int j = 0; j < k; ++j) {
        float bv = -INFINITY;
        int bi = 0x7fffffff;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            int e = lane + 32 * i;
            if (e < E && (v[i] > bv || (v[i] == bv && e < bi))) { bv = v[i]; bi = e; }
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
        if ((bi & 31) == lane) {
#pragma unroll
            for (int i = 0; i < 8; ++i)
                if (i == (bi >> 5)) v[i] = -INFINITY;   // taken; E real logits are finite
        }
    }
    if (lane < k) {
        const float Z = renorm ? zsel : zall;
        idx[(int64_t)t * k + lane] = my_idx;
        w[(int64_t)t * k + lane] = expf(my_val - m) / Z;
    }
}

}  // namespace

int32_t efk_route_topk(ef_ctx* ctx, cudaStream_t st, const void* x, const void* wr, const float* bias,
                       int64_t bias_stride, int T, int renorm, int32_t* idx, float* w, float* logits) {
    if (T == 0) return EF_OK;
    const int E = ctx->cfg.n_experts, d = ctx->cfg.d_model, k = ctx->cfg.top_k;
    dim3 grid((T + kWarps - 1) / kWarps), block(kWarps * 32);
    size_t smem = (size_t)kWarps * E * sizeof(float);
    route_topk_kernel<<<grid, block, smem, st>>>((const uint4*)x, (const uint4*)wr, bias, bias_stride, T, d / 8, E, k,
                                                 renorm, idx, w, logits);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    return EF_OK;
}
