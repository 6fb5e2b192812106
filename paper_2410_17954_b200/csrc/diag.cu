// Diagnostics that are not on the hot path.  libef_diag only (include/ef_diag.h).
//
// ef_diag_tma_fill_gbs: how fast TMA can fill shared memory on this device.  The grouped GEMM (ffn_tc.cu) stages
// 48 KB of operands per CTA per k-block (1024 tensor cycles at full rate), i.e. it asks the L2 -> SM path for 48 bytes
// per clock and SM; how close that is to what the device can deliver decides whether the tensor pipe can be kept fed
// (contiguous 32 KB boxes fill at 18-21 TB/s, the same box gathered from 256 strided rows at
// 14 TB/s -- the reason the packed expert layout is tiled).  This kernel measures the ceiling directly: one persistent
// CTA per SM, one producer lane streaming 32 KB boxes (the GEMM's weight box: 256 rowlets x 64 bf16, 128-byte
// swizzle) through a 4-stage ring, one consumer lane freeing them; CTA-scope barriers only.
#include <algorithm>

#include "ef_internal.h"
#include "ef_diag.h"

namespace {

constexpr int kStages = 4;
constexpr int BOX_ROWS = 256, BOX_COLS = 64;
constexpr int BOX_BYTES = BOX_ROWS * BOX_COLS * 2;

struct Ctl { uint64_t full[kStages]; uint64_t empty[kStages]; };
constexpr size_t kSmem = 1024 + (size_t)kStages * BOX_BYTES + sizeof(Ctl);

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

__global__ void __launch_bounds__(64, 1) tma_fill_kernel(const __grid_constant__ CUtensorMap tm, int iters, int n_boxes) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    Ctl* ctl = (Ctl*)(smem + (size_t)kStages * BOX_BYTES);
    if (threadIdx.x == 0) {
        for (int i = 0; i < kStages; ++i) { mbar_init(&ctl->full[i], 1); mbar_init(&ctl->empty[i], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int stage = 0; uint32_t phase = 0;
        for (int i = 0; i < iters; ++i) {
            mbar_wait(&ctl->empty[stage], phase ^ 1);
            mbar_expect_tx(&ctl->full[stage], BOX_BYTES);
            const int box = (int)(((long long)blockIdx.x * iters + i) % n_boxes);      // every CTA its own boxes
            asm volatile(
                "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
                ::"r"(smem_u32(smem + (size_t)stage * BOX_BYTES)), "l"(&tm), "r"(smem_u32(&ctl->full[stage])), "r"(0),
                  "r"(box * BOX_ROWS) : "memory");
            if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
    } else if (threadIdx.x == 32) {
        int stage = 0; uint32_t phase = 0;
        for (int i = 0; i < iters; ++i) {
            mbar_wait(&ctl->full[stage], phase);
            mbar_arrive(&ctl->empty[stage]);
            if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
    }
}


// ef_diag_pair_handoff_gbs: the same stream run by CTA PAIRS the way the grouped GEMM runs it -- both CTAs' boxes complete
// on the LEADER's "full" barrier, the leader's consumer lane hands each stage back to both producers -- with the hand-back
// to the peer either a cluster-scope RELEASE arrive (mode 0) or a RELAXED one (mode 1).  The consumer has written nothing
// the producer reads, so relaxed is enough; the release costs a MEMBAR.GPU per stage.  (Measured on a B200, 16 CTAs, boxes
// out of HBM: 33 GB/s per SM with the release, 111 GB/s relaxed, 139 GB/s for the unpaired stream above.)
__device__ __forceinline__ uint32_t mapa_u32(const void* p, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(p)), "r"(rank));
    return r;
}
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(64, 1) pair_handoff_kernel(const __grid_constant__ CUtensorMap tm, int iters,
                                                                                        int n_boxes, int relaxed) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    Ctl* ctl = (Ctl*)(smem + (size_t)kStages * BOX_BYTES);
    uint32_t rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    if (threadIdx.x == 0) {
        for (int i = 0; i < kStages; ++i) { mbar_init(&ctl->full[i], 1); mbar_init(&ctl->empty[i], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    if (threadIdx.x == 0) {                                   // producer of either CTA
        int stage = 0; uint32_t phase = 0;
        for (int i = 0; i < iters; ++i) {
            mbar_wait(&ctl->empty[stage], phase ^ 1);
            if (rank == 0) mbar_expect_tx(&ctl->full[stage], 2 * BOX_BYTES);
            const int box = (int)(((long long)blockIdx.x * iters + i) % n_boxes);
            asm volatile(
                "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.cta_group::2 [%0], [%1, {%3, %4}], [%2];"
                ::"r"(smem_u32(smem + (size_t)stage * BOX_BYTES)), "l"(&tm), "r"(mapa_u32(&ctl->full[stage], 0)), "r"(0),
                  "r"(box * BOX_ROWS) : "memory");
            if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
    } else if (threadIdx.x == 32 && rank == 0) {              // the leader's consumer
        int stage = 0; uint32_t phase = 0;
        for (int i = 0; i < iters; ++i) {
            mbar_wait(&ctl->full[stage], phase);
            mbar_arrive(&ctl->empty[stage]);
            const uint32_t peer = mapa_u32(&ctl->empty[stage], 1);
            if (relaxed) asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(peer) : "memory");
            else asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(peer) : "memory");
            if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
    }
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");     // the peer's barriers stay alive until both are done
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

// mode < 0: the unpaired stream on `grid` CTAs; mode 0 / 1: the pair stream with a release / relaxed hand-back
static int32_t run_fill(ef_ctx* ctx, const char* who, int64_t region_bytes, int32_t iters, int grid, int mode, double* gbs_out) {
    if (!gbs_out || iters < 1 || region_bytes < BOX_BYTES || grid < 1 || grid > ctx->n_sms || (mode >= 0 && (grid & 1)))
        return ef_fail(ctx, EF_ERR_INVALID_ARG, "%s: need gbs_out, iters >= 1, region_bytes >= %d, 1 <= CTAs <= SM count (even for pairs)",
                       who, BOX_BYTES);
    void* fp = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
        return ef_fail(ctx, EF_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    const int n_boxes = (int)std::min<int64_t>(region_bytes / BOX_BYTES, 1 << 20);
    void* buf = nullptr;
    cudaError_t e = cudaMalloc(&buf, (size_t)n_boxes * BOX_BYTES);
    if (e != cudaSuccess) return ef_fail(ctx, EF_ERR_OOM, "%s: scratch region: %s", who, cudaGetErrorString(e));
    int32_t rc = EF_OK;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    do {
        if ((e = cudaMemset(buf, 0, (size_t)n_boxes * BOX_BYTES)) != cudaSuccess) break;
        CUtensorMap tm;
        cuuint64_t dims[2] = {BOX_COLS, (cuuint64_t)n_boxes * BOX_ROWS};
        cuuint64_t strides[1] = {BOX_COLS * 2};
        cuuint32_t box[2] = {BOX_COLS, BOX_ROWS};
        cuuint32_t estr[2] = {1, 1};
        CUresult r = ((EncodeTiledFn)fp)(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, buf, dims, strides, box, estr,
                                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { rc = ef_fail(ctx, EF_ERR_CUDA, "cuTensorMapEncodeTiled failed: %d", (int)r); break; }
        if ((e = cudaFuncSetAttribute(tma_fill_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem)) != cudaSuccess) break;
        if ((e = cudaFuncSetAttribute(pair_handoff_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem)) != cudaSuccess) break;
        if ((e = cudaEventCreate(&e0)) != cudaSuccess || (e = cudaEventCreate(&e1)) != cudaSuccess) break;
        float best = 0.f;
        for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {       // first pass warms L2; best of the rest
            cudaEventRecord(e0, 0);
            if (mode < 0) tma_fill_kernel<<<grid, 64, kSmem, 0>>>(tm, iters, n_boxes);
            else pair_handoff_kernel<<<grid, 64, kSmem, 0>>>(tm, iters, n_boxes, mode);
            cudaEventRecord(e1, 0);
            if ((e = cudaEventSynchronize(e1)) != cudaSuccess) break;
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && (best == 0.f || ms < best)) best = ms;
            ctx->launches++;
        }
        if (e == cudaSuccess && best > 0.f) *gbs_out = (double)grid * iters * BOX_BYTES / (best * 1e-3) / 1e9;
    } while (0);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess) { ctx->sticky = EF_ERR_CUDA; return ef_fail(ctx, EF_ERR_CUDA, "%s: %s", who, cudaGetErrorString(e)); }
    return rc;
}

extern "C" int32_t ef_diag_tma_fill_gbs(ef_ctx* ctx, int64_t region_bytes, int32_t iters, double* gbs_out) {
    EF_CHECK_CTX(ctx);
    return run_fill(ctx, "ef_diag_tma_fill_gbs", region_bytes, iters, ctx->n_sms, -1, gbs_out);
}

extern "C" int32_t ef_diag_pair_handoff_gbs(ef_ctx* ctx, int64_t region_bytes, int32_t iters, int32_t n_ctas, int32_t mode,
                                            double* gbs_out) {
    EF_CHECK_CTX(ctx);
    if (mode < -1 || mode > 1) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_diag_pair_handoff_gbs: mode is -1, 0 or 1");
    return run_fill(ctx, "ef_diag_pair_handoff_gbs", region_bytes, iters, n_ctas, mode, gbs_out);
}
