// a5: combine (Eq. 2, summed over the k selected experts) and a8: RMSNorm (cfg 5).
//
// Both HBM-bound.  combine reads 2*d*k bytes per token (+ residual, + shared rows) and writes 2*d;
// one thread per 8 columns, 128-bit loads, fp32 accumulate, ONE rounding to bf16 (error budget,
// DESIGN.md §6).  rmsnorm: one CTA per token, row kept in registers between the two passes.
#include <cuda_bf16.h>

#include "ef_internal.h"

namespace {

__device__ __forceinline__ float bf_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);   // .x = lo (low 16 bits), round-to-nearest-even
    return *reinterpret_cast<uint32_t*>(&v);
}

__device__ __forceinline__ void fma8(float* acc, const uint4& v, float s) {
    acc[0] = fmaf(s, bf_lo(v.x), acc[0]); acc[1] = fmaf(s, bf_hi(v.x), acc[1]);
    acc[2] = fmaf(s, bf_lo(v.y), acc[2]); acc[3] = fmaf(s, bf_hi(v.y), acc[3]);
    acc[4] = fmaf(s, bf_lo(v.z), acc[4]); acc[5] = fmaf(s, bf_hi(v.z), acc[5]);
    acc[6] = fmaf(s, bf_lo(v.w), acc[6]); acc[7] = fmaf(s, bf_hi(v.w), acc[7]);
}

__global__ void __launch_bounds__(256)
combine_kernel(const uint4* __restrict__ y_perm, const int32_t* __restrict__ inv, const float* __restrict__ w,
               int T, int k, int d8, int n_shared, const uint4* __restrict__ residual,
               const uint4* __restrict__ y_shared, uint4* __restrict__ out) {
    const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (int64_t)T * d8) return;
    const int t = (int)(gid / d8), c = (int)(gid % d8);
    float acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = 0.f;
    if (residual) fma8(acc, residual[gid], 1.f);
    for (int j = 0; j < k; ++j) {
        const int row = inv[t * k + j];
        const float s = w[t * k + j];
        if (row >= 0) fma8(acc, y_perm[(int64_t)row * d8 + c], s);      // -1: a pair ef_permute could not route
    }
    for (int s = 0; s < n_shared; ++s) fma8(acc, y_shared[((int64_t)s * T + t) * d8 + c], 1.f);
    uint4 o;
    o.x = pack_bf16(acc[0], acc[1]); o.y = pack_bf16(acc[2], acc[3]);
    o.z = pack_bf16(acc[4], acc[5]); o.w = pack_bf16(acc[6], acc[7]);
    out[gid] = o;
}

constexpr int kNormThreads = 256;
constexpr int kNormCache = 4;   // uint4 per thread kept in registers: rows up to 8192 columns

__global__ void __launch_bounds__(kNormThreads)
rmsnorm_kernel(const uint4* __restrict__ x, int d8, int d, float eps, uint4* __restrict__ out) {
    __shared__ float s_part[kNormThreads / 32];
    const uint4* xr = x + (int64_t)blockIdx.x * d8;
    uint4* orow = out + (int64_t)blockIdx.x * d8;
    uint4 cache[kNormCache];
    float ss = 0.f;
#pragma unroll
    for (int i = 0; i < kNormCache; ++i) {
        const int c = threadIdx.x + i * kNormThreads;
        if (c < d8) {
            const uint4 v = xr[c];
            cache[i] = v;
            float a[8] = {bf_lo(v.x), bf_hi(v.x), bf_lo(v.y), bf_hi(v.y), bf_lo(v.z), bf_hi(v.z), bf_lo(v.w), bf_hi(v.w)};
#pragma unroll
            for (int q = 0; q < 8; ++q) ss = fmaf(a[q], a[q], ss);
        }
    }
    for (int c = threadIdx.x + kNormCache * kNormThreads; c < d8; c += kNormThreads) {
        const uint4 v = xr[c];
        float a[8] = {bf_lo(v.x), bf_hi(v.x), bf_lo(v.y), bf_hi(v.y), bf_lo(v.z), bf_hi(v.z), bf_lo(v.w), bf_hi(v.w)};
#pragma unroll
        for (int q = 0; q < 8; ++q) ss = fmaf(a[q], a[q], ss);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = ss;
    __syncthreads();
    float tot = 0.f;
#pragma unroll
    for (int i = 0; i < kNormThreads / 32; ++i) tot += s_part[i];
    const float scale = 1.0f / sqrtf(tot / (float)d + eps);
    auto emit = [&](const uint4& v, int c) {
        uint4 o;
        o.x = pack_bf16(bf_lo(v.x) * scale, bf_hi(v.x) * scale);
        o.y = pack_bf16(bf_lo(v.y) * scale, bf_hi(v.y) * scale);
        o.z = pack_bf16(bf_lo(v.z) * scale, bf_hi(v.z) * scale);
        o.w = pack_bf16(bf_lo(v.w) * scale, bf_hi(v.w) * scale);
        orow[c] = o;
    };
#pragma unroll
    for (int i = 0; i < kNormCache; ++i) {
        const int c = threadIdx.x + i * kNormThreads;
        if (c < d8) emit(cache[i], c);
    }
    for (int c = threadIdx.x + kNormCache * kNormThreads; c < d8; c += kNormThreads) emit(xr[c], c);
}

}  // namespace

int32_t efk_combine(ef_ctx* ctx, cudaStream_t st, const void* y_perm, const int32_t* inv, const float* w, int T,
                    const void* residual, const void* y_shared, void* out) {
    if (T == 0) return EF_OK;
    const int d8 = ctx->cfg.d_model / 8, k = ctx->cfg.top_k;
    const int64_t n = (int64_t)T * d8;
    const int blocks = (int)((n + 255) / 256);
    combine_kernel<<<blocks, 256, 0, st>>>((const uint4*)y_perm, inv, w, T, k, d8, y_shared ? ctx->cfg.n_shared : 0,
                                           (const uint4*)residual, (const uint4*)y_shared, (uint4*)out);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    return EF_OK;
}

int32_t efk_rmsnorm(ef_ctx* ctx, cudaStream_t st, const void* x, int T, float eps, void* out) {
    if (T == 0) return EF_OK;
    const int d = ctx->cfg.d_model;
    rmsnorm_kernel<<<T, kNormThreads, 0, st>>>((const uint4*)x, d / 8, d, eps, (uint4*)out);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    return EF_OK;
}
