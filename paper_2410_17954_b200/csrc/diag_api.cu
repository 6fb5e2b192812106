// libef_diag only (include/ef_diag.h): the bring-up and probing hooks.  None of this is compiled into libef.so.
#include "ef_internal.h"
#include "ef_diag.h"

extern "C" int32_t ef_diag_set_simt_ffn(ef_ctx* ctx, int32_t on) {
    EF_CHECK_CTX(ctx);
    ctx->debug_simt = on ? 1 : 0;
    return EF_OK;
}

// -DEF_KPROF builds only: per-CTA {total, wait ticket, wait TMEM, wait TMA, units} cycles of the MMA-issuing lane for the
// last launch that ran GEMM1 units (which = 1) or only GEMM2 units (which = 2).  out: HOST int64[n_sms * 5].  Synchronous.
extern "C" int32_t ef_diag_kprof(ef_ctx* ctx, int32_t which, int64_t* out) {
    EF_CHECK_CTX(ctx);
#ifdef EF_KPROF
    if (!out || (which != 1 && which != 2)) return ef_fail(ctx, EF_ERR_INVALID_ARG, "ef_diag_kprof: bad argument");
    const size_t bytes = sizeof(long long) * 5 * (size_t)ctx->n_sms;
    for (long long** p : {&ctx->kprof1, &ctx->kprof2})
        if (!*p) { EF_CUDA(ctx, cudaMalloc(p, bytes)); EF_CUDA(ctx, cudaMemset(*p, 0, bytes)); }
    EF_CUDA(ctx, cudaDeviceSynchronize());
    EF_CUDA(ctx, cudaMemcpy(out, which == 1 ? ctx->kprof1 : ctx->kprof2, bytes, cudaMemcpyDeviceToHost));
    return EF_OK;
#else
    (void)which; (void)out;
    return ef_fail(ctx, EF_ERR_UNSUPPORTED, "ef_diag_kprof: library built without -DEF_KPROF");
#endif
}
