// Plain-FMA grouped SwiGLU FFN.  BRING-UP AID ONLY, libef_diag only (ef_diag_set_simt_ffn): a second, simple CUDA
// implementation of a4 used to triangulate the tcgen05 kernels on the device.  Not the product path,
// never selected automatically.  Reads the same packed expert layout (ef_internal.h).
#include <cuda_bf16.h>

#include "ef_internal.h"

namespace {

constexpr int TM = 64, TN = 64, TK = 16;

__device__ __forceinline__ float bf2f(uint16_t b) { return __uint_as_float(((uint32_t)b) << 16); }

struct SimtGroup { int32_t a_row0, c_row0, rows, slot; };
struct SimtTable { int32_t n; SimtGroup g[EF_MAX_GROUPS]; };

__device__ __forceinline__ bool find_tile(const SimtTable& tab, int tile, int& g, int& mt) {
    for (int i = 0; i < tab.n; ++i) {
        int nt = (tab.g[i].rows + TM - 1) / TM;
        if (tile < nt) { g = i; mt = tile; return true; }
        tile -= nt;
    }
    return false;
}

// C[m, n] for 64x64 tile; A rows from `a` (ld = K), B rows given by functor rowptr(n) (K-major).
template <int kEpi>     // 0 plain, 1 SwiGLU (packed gate/up rows), 2 ReLU
__global__ void __launch_bounds__(256)
simt_gemm_kernel(const uint16_t* __restrict__ a, uint16_t* __restrict__ c, const char* __restrict__ arena, int64_t W,
                 int64_t b_off_bytes, int K, int N, int b_rows, SimtTable tab) {
    constexpr bool kSwiglu = kEpi == 1;
    __shared__ float As[TK][TM + 1];
    __shared__ float B0[TK][TN + 1];
    __shared__ float B1[kSwiglu ? TK : 1][TN + 1];
    int g, mt;
    if (!find_tile(tab, blockIdx.y, g, mt)) return;
    const SimtGroup grp = tab.g[g];
    const int rows = grp.rows;
    const int m0 = mt * TM, n0 = blockIdx.x * TN;
    const uint16_t* A = a + (int64_t)grp.a_row0 * K;
    const uint16_t* Bbase = (const uint16_t*)(arena + (int64_t)grp.slot * W + b_off_bytes);
    uint16_t* C = c + (int64_t)grp.c_row0 * N;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    float acc0[4][4] = {}, acc1[4][4] = {};
    for (int k0 = 0; k0 < K; k0 += TK) {
        for (int i = threadIdx.x; i < TM * TK; i += 256) {
            int r = i / TK, kk = i % TK;
            int m = m0 + r;
            As[kk][r] = (m < rows) ? bf2f(A[(int64_t)m * K + k0 + kk]) : 0.f;
            int n = n0 + r;   // TN == TM
            if (kSwiglu) {
                // h column n -> gate row 256*(n/128) + n%128, up row = gate row + 128
                int64_t gr = (int64_t)(n / EF_W13_BLOCK) * (2 * EF_W13_BLOCK) + (n % EF_W13_BLOCK);
                B0[kk][r] = (n < N) ? bf2f(Bbase[ef_tiled_index(gr, k0 + kk, b_rows, K)]) : 0.f;
                B1[kk][r] = (n < N) ? bf2f(Bbase[ef_tiled_index(gr + EF_W13_BLOCK, k0 + kk, b_rows, K)]) : 0.f;
            } else {
                B0[kk][r] = (n < N) ? bf2f(Bbase[ef_tiled_index(n, k0 + kk, b_rows, K)]) : 0.f;
            }
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < TK; ++kk) {
            float av[4], b0[4], b1[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) av[i] = As[kk][ty * 4 + i];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                b0[j] = B0[kk][tx * 4 + j];
                b1[j] = kSwiglu ? B1[kk][tx * 4 + j] : 0.f;
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    acc0[i][j] = fmaf(av[i], b0[j], acc0[i][j]);
                    if (kSwiglu) acc1[i][j] = fmaf(av[i], b1[j], acc1[i][j]);
                }
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        int m = m0 + ty * 4 + i;
        if (m >= rows) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int n = n0 + tx * 4 + j;
            if (n >= N) continue;
            float v = acc0[i][j];
            if (kSwiglu) v = v / (1.f + expf(-v)) * acc1[i][j];
            if (kEpi == 2) v = fmaxf(v, 0.f);
            __nv_bfloat16 o = __float2bfloat16_rn(v);
            C[(int64_t)m * N + n] = *reinterpret_cast<uint16_t*>(&o);
        }
    }
}

}  // namespace

int32_t efk_ffn_simt(ef_ctx* ctx, cudaStream_t st, const void* x, void* y, const EfWaveTable& tab, int phase) {
    const int d = ctx->cfg.d_model, f = ctx->cfg.d_ff;
    int tiles = 0;
    SimtTable t1, t2;
    t1.n = t2.n = tab.n;
    for (int i = 0; i < tab.n; ++i) {
        tiles += (tab.g[i].rows + TM - 1) / TM;
        t1.g[i] = SimtGroup{tab.g[i].x_row0, tab.g[i].h_row0, tab.g[i].rows, tab.g[i].slot};   // GEMM1: x rows -> h rows
        t2.g[i] = SimtGroup{tab.g[i].h_row0, tab.g[i].y_row0, tab.g[i].rows, tab.g[i].slot};   // GEMM2: h rows -> y rows
    }
    if (tiles == 0) return EF_OK;
    const bool relu = ctx->cfg.expert_kind == 1;
    if (phase & 1) {
        if (relu)
            simt_gemm_kernel<2><<<dim3((f + TN - 1) / TN, tiles), 256, 0, st>>>(
                (const uint16_t*)x, (uint16_t*)ctx->h_ws, ctx->arena, ctx->W, 0, d, f, f, t1);
        else
            simt_gemm_kernel<1><<<dim3((f + TN - 1) / TN, tiles), 256, 0, st>>>(
                (const uint16_t*)x, (uint16_t*)ctx->h_ws, ctx->arena, ctx->W, 0, d, f, 2 * f, t1);
        ctx->launches++;
    }
    if (phase & 2) {
        simt_gemm_kernel<0><<<dim3((d + TN - 1) / TN, tiles), 256, 0, st>>>(
            (const uint16_t*)ctx->h_ws, (uint16_t*)y, ctx->arena, ctx->W, (int64_t)(relu ? 1 : 2) * f * d * 2, f, d, d, t2);
        ctx->launches++;
    }
    EF_CUDA(ctx, cudaGetLastError());
    return EF_OK;
}
