/*
 * ef_diag.h -- extra entry points of libef_diag.so, the DIAGNOSTIC build of libef (same sources compiled with -DEF_DIAG
 * plus csrc/ffn_simt.cu, csrc/diag.cu, csrc/diag_api.cu; `python -m paper_2410_17954_b200.build --diag`).
 * libef_diag.so exports everything ef.h declares and, in addition, the bring-up and probing hooks below.  None of them
 * exists in libef.so: the product library has ONE grouped-FFN backend (csrc/ffn_tc.cu) and no probe kernels.
 */
#ifndef EF_DIAG_H_
#define EF_DIAG_H_

#include "ef.h"

#ifdef __cplusplus
extern "C" {
#endif

/* 0 = tcgen05 kernels (default); 1 = plain-FMA kernels for the grouped FFN (csrc/ffn_simt.cu): a second, simple CUDA
 * implementation used to triangulate the tcgen05 path on the device during bring-up.  Slow. */
int32_t ef_diag_set_simt_ffn(ef_ctx* ctx, int32_t on);
/* The rate at which TMA can fill shared memory on this device, i.e. the L2 -> SM fabric ceiling that bounds the grouped
 * GEMM's operand traffic.  One persistent CTA per SM streams 32 KB boxes (64 x 256 bf16, the GEMM's
 * weight box) through a 4-stage ring, `iters` boxes per CTA, out of a scratch region of region_bytes (<= 126 MB stays in
 * L2; larger streams from HBM).  gbs_out: HOST double, delivered GB/s.  Synchronous; allocates and frees the region. */
int32_t ef_diag_tma_fill_gbs(ef_ctx* ctx, int64_t region_bytes, int32_t iters, double* gbs_out);
/* What a cross-CTA hand-back costs on this device ("hand-overs"): n_ctas CTAs (1..SM count; even for the
 * pair modes) stream the same boxes; mode -1: every CTA on its own (the stream above on fewer SMs); mode 0 / 1: CTA PAIRS
 * (clusters of 2) run the grouped GEMM's protocol -- both CTAs' boxes complete on the leader's barrier, the leader's
 * consumer lane hands each stage back to the peer's producer with a remote mbarrier arrive that is a cluster-scope
 * RELEASE (0) or RELAXED (1).  The release is a MEMBAR.GPU per stage and throttles the stream to about a third.
 * gbs_out: HOST double, delivered GB/s over all n_ctas.  Synchronous; allocates and frees the region. */
int32_t ef_diag_pair_handoff_gbs(ef_ctx* ctx, int64_t region_bytes, int32_t iters, int32_t n_ctas, int32_t mode, double* gbs_out);
/* Only in a diag library built with -DEF_KPROF as well (EF_ERR_UNSUPPORTED otherwise): the first call arms the counters,
 * later calls return, per CTA pair of the last launch that ran GEMM1 units (which = 1) or only GEMM2 units (which = 2),
 * the cycles the MMA-issuing lane spent {in total, waiting for a tile ticket, waiting for the epilogue to free TMEM,
 * waiting for TMA to fill a stage} and the units it processed.  out: HOST int64[5 * SM count].  Synchronous. */
int32_t ef_diag_kprof(ef_ctx* ctx, int32_t which, int64_t* out);

#ifdef __cplusplus
}
#endif
#endif /* EF_DIAG_H_ */
