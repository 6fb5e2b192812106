/*
 * moe_oracle.c -- CPU ORACLE for the ExpertFlow MoE expert layer.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  The product path (paper_2410_17954_b200/) never does, and the
 * two share no code.
 *
 * What it is: the plain definition of what the layer computes, written as
 * loops a reader can check against the paper by eye.  Inputs are bf16 bit patterns, widened
 * exactly; all arithmetic is in `real` (double by default; -DORC_REAL=float builds the fp32
 * variant BASELINE.json's north_star mentions, used only to show the fp32-vs-fp64 gap).
 * No blocking, no fusion, no intermediate rounding.  The only liberty: the summation order
 * inside one dot product is left to the compiler (omp simd reduction), which in fp64 changes
 * results by ~1e-16 relative.
 *
 * Citations: P:L<n> = /root/reference/PAPER.md line n.
 *   gate            Eq. 1
 *   selection/out   Eq. 2, P:L44-46 (top-1; generalised to top-k per P:L52 "top-k highest weights")
 *   dispatch        implied P:L21, P:L68 ("each expert processes only a few tokens")
 *   expert e_i      opaque at P:L46; SwiGLU without biases is BASELINE.json's choice (R4)
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): numpy fp64 matmul+softmax; brute-force top-k with
 * exact ties; permutation bijection / counts / stability; identical experts == one dense SwiGLU
 * FFN (numpy); k=1,renorm=0 == Eq. 2; linearity of combine; fp32 build vs fp64 build.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef ORC_REAL
#define ORC_REAL double
#endif
typedef ORC_REAL real;

#if defined(_OPENMP)
#include <omp.h>
#endif

/* exact bf16 -> real */
static inline real bf16_to_real(uint16_t b) {
    union { uint32_t u; float f; } c;
    c.u = ((uint32_t)b) << 16;
    return (real)c.f;
}

static inline real dot_bf16(const uint16_t* a, const uint16_t* b, int64_t n) {
    real acc = 0;
#pragma omp simd reduction(+ : acc)
    for (int64_t i = 0; i < n; ++i) acc += bf16_to_real(a[i]) * bf16_to_real(b[i]);
    return acc;
}

static inline real dot_real_bf16(const real* a, const uint16_t* b, int64_t n) {
    real acc = 0;
#pragma omp simd reduction(+ : acc)
    for (int64_t i = 0; i < n; ++i) acc += a[i] * bf16_to_real(b[i]);
    return acc;
}

int orc_real_bytes(void) { return (int)sizeof(real); }

int orc_num_threads(void) {
#if defined(_OPENMP)
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Eq. 1 numerator argument: l[t,e] = w_e . x_t + b_e.
 * bias may be NULL; bias_token_stride = 0 (per-expert bias [E]) or E (per-token bias [T,E]). */
void orc_router_logits(const uint16_t* x, const uint16_t* wr, const float* bias, int64_t bias_token_stride,
                       int T, int d, int E, real* logits /*[T,E]*/) {
#pragma omp parallel for schedule(static)
    for (int t = 0; t < T; ++t)
        for (int e = 0; e < E; ++e) {
            real b = bias ? (real)bias[(int64_t)t * bias_token_stride + e] : (real)0;
            logits[(int64_t)t * E + e] = b + dot_bf16(x + (int64_t)t * d, wr + (int64_t)e * d, d);
        }
}

/* Top-k selection (Eq. 2's argmax repeated k times; ties -> smallest expert index) and gate
 * weights.  renorm=1: softmax over the k selected logits; renorm=0: Eq. 1's full softmax
 * probability of each selected expert.  idx/w are in pick order (descending logit). */
void orc_topk_gate(const real* logits, int T, int E, int k, int renorm, int32_t* idx /*[T,k]*/, real* w /*[T,k]*/) {
    for (int t = 0; t < T; ++t) {
        const real* l = logits + (int64_t)t * E;
        char* taken = (char*)calloc((size_t)E, 1);
        for (int j = 0; j < k; ++j) {
            int best = -1;
            for (int e = 0; e < E; ++e) {
                if (taken[e]) continue;
                if (best < 0 || l[e] > l[best]) best = e; /* strict > keeps the smaller index on ties */
            }
            taken[best] = 1;
            idx[(int64_t)t * k + j] = best;
        }
        free(taken);
        real m = l[0];
        for (int e = 1; e < E; ++e)
            if (l[e] > m) m = l[e];
        real Z = 0;
        if (renorm) {
            for (int j = 0; j < k; ++j) Z += exp((double)(l[idx[(int64_t)t * k + j]] - m));
        } else {
            for (int e = 0; e < E; ++e) Z += exp((double)(l[e] - m));
        }
        for (int j = 0; j < k; ++j) w[(int64_t)t * k + j] = (real)exp((double)(l[idx[(int64_t)t * k + j]] - m)) / Z;
    }
}

/* Dispatch: stable counting sort of the flat (token, choice) pairs p = t*k + j by expert id.
 * counts[E], offsets[E+1] (exclusive prefix), inv[p] = row, src[row] = p. */
void orc_permute(const int32_t* idx, int T, int k, int E, int32_t* counts, int32_t* offsets, int32_t* src,
                 int32_t* inv) {
    int64_t R = (int64_t)T * k;
    for (int e = 0; e < E; ++e) counts[e] = 0;
    for (int64_t p = 0; p < R; ++p) counts[idx[p]]++;
    offsets[0] = 0;
    for (int e = 0; e < E; ++e) offsets[e + 1] = offsets[e] + counts[e];
    int32_t* seen = (int32_t*)calloc((size_t)E, sizeof(int32_t));
    for (int64_t p = 0; p < R; ++p) {
        int e = idx[p];
        int32_t row = offsets[e] + seen[e]++;
        inv[p] = row;
        src[row] = (int32_t)p;
    }
    free(seen);
}

/* x_perm[row,:] = x[src[row] / k, :]  (bf16 copy) */
void orc_gather_rows(const uint16_t* x, const int32_t* src, int64_t R, int k, int d, uint16_t* x_perm) {
    for (int64_t r = 0; r < R; ++r) memcpy(x_perm + r * d, x + (int64_t)(src[r] / k) * d, (size_t)d * 2);
}

/* One expert e_i applied to M rows: SwiGLU FFN without biases.
 *   g_n = sum_d x[r,d] Wg[n,d];  u_n = sum_d x[r,d] Wu[n,d];  h_n = g_n / (1 + exp(-g_n)) * u_n
 *   y[r,c] = sum_n h_n Wd[c,n]
 * xrows: [M, d] bf16; wg, wu: [f, d] bf16; wd: [d, f] bf16; y: [M, d] real; h_out (nullable): [M, f]. */
void orc_expert_ffn(const uint16_t* xrows, int64_t M, int d, int f, const uint16_t* wg, const uint16_t* wu,
                    const uint16_t* wd, real* y, real* h_out) {
#pragma omp parallel
    {
        real* h = (real*)malloc((size_t)f * sizeof(real));
#pragma omp for schedule(dynamic, 1)
        for (int64_t r = 0; r < M; ++r) {
            const uint16_t* xr = xrows + r * d;
            for (int n = 0; n < f; ++n) {
                real g = dot_bf16(xr, wg + (int64_t)n * d, d);
                real u = dot_bf16(xr, wu + (int64_t)n * d, d);
                h[n] = g / ((real)1 + (real)exp(-(double)g)) * u;
            }
            if (h_out) memcpy(h_out + r * f, h, (size_t)f * sizeof(real));
            for (int c = 0; c < d; ++c) y[r * d + c] = dot_real_bf16(h, wd + (int64_t)c * f, f);
        }
        free(h);
    }
}

/* Switch-style expert (R30): the non-gated ReLU FFN of the Switch / T5 models the paper evaluates,
 * without biases:  h_n = max(0, sum_d x[r,d] W1[n,d]);  y[r,c] = sum_n h_n W2[c,n].
 * xrows: [M, d] bf16; w1: [f, d] bf16; w2: [d, f] bf16; y: [M, d] real; h_out (nullable): [M, f]. */
void orc_expert_ffn_relu(const uint16_t* xrows, int64_t M, int d, int f, const uint16_t* w1, const uint16_t* w2,
                         real* y, real* h_out) {
#pragma omp parallel
    {
        real* h = (real*)malloc((size_t)f * sizeof(real));
#pragma omp for schedule(dynamic, 1)
        for (int64_t r = 0; r < M; ++r) {
            const uint16_t* xr = xrows + r * d;
            for (int n = 0; n < f; ++n) {
                real a = dot_bf16(xr, w1 + (int64_t)n * d, d);
                h[n] = a > (real)0 ? a : (real)0;
            }
            if (h_out) memcpy(h_out + r * f, h, (size_t)f * sizeof(real));
            for (int c = 0; c < d; ++c) y[r * d + c] = dot_real_bf16(h, w2 + (int64_t)c * f, f);
        }
        free(h);
    }
}

/* Combine (Eq. 2 summed over the k selected experts):
 *   out[t,c] = res[t,c] + sum_j w[t,j] * y_perm[inv[t*k+j], c] + y_shared[t,c]
 * res (bf16, nullable), y_shared (real, nullable). */
void orc_combine(const real* y_perm, const int32_t* inv, const real* w, int T, int k, int d, const uint16_t* res,
                 const real* y_shared, real* out) {
#pragma omp parallel for schedule(static)
    for (int t = 0; t < T; ++t)
        for (int c = 0; c < d; ++c) {
            real acc = res ? bf16_to_real(res[(int64_t)t * d + c]) : (real)0;
            for (int j = 0; j < k; ++j)
                acc += w[(int64_t)t * k + j] * y_perm[(int64_t)inv[(int64_t)t * k + j] * d + c];
            if (y_shared) acc += y_shared[(int64_t)t * d + c];
            out[(int64_t)t * d + c] = acc;
        }
}

/* RMSNorm with unit gain (BASELINE.json cfg 5; R19): u = x / sqrt(mean(x^2) + eps). */
void orc_rmsnorm(const uint16_t* x, int T, int d, double eps, real* out) {
    for (int t = 0; t < T; ++t) {
        real ss = 0;
        for (int c = 0; c < d; ++c) {
            real v = bf16_to_real(x[(int64_t)t * d + c]);
            ss += v * v;
        }
        real s = (real)1 / (real)sqrt((double)(ss / (real)d) + eps);
        for (int c = 0; c < d; ++c) out[(int64_t)t * d + c] = bf16_to_real(x[(int64_t)t * d + c]) * s;
    }
}

/* real -> bf16 bits, round to nearest even (used to hand a layer's output to the next layer in
 * the cfg-5 stack exactly as the boundary defines it: activations between calls are bf16). */
void orc_round_bf16(const real* a, int64_t n, uint16_t* out) {
    for (int64_t i = 0; i < n; ++i) {
        union { uint32_t u; float f; } c;
        c.f = (float)a[i];
        uint32_t u = c.u;
        if ((u & 0x7F800000u) == 0x7F800000u && (u & 0x007FFFFFu)) { out[i] = (uint16_t)((u >> 16) | 0x40); continue; }
        u += 0x7FFFu + ((u >> 16) & 1u);
        out[i] = (uint16_t)(u >> 16);
    }
}
