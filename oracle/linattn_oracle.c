/*
 * ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares no code with the CUDA path.
 *
 * Gated linear-attention recurrence, written out as its plain definition in fp64.
 *
 * Source of the definition: BASELINE.json `north_star` ("the sequential recurrence
 * S_t = g_t·S_{t-1} + k_tᵀ v_t, o_t = q_t·S_t"), SURVEY.md §8(c) "Definition".
 * PAPER.md never prints the recurrence: it only says the linear-attention state is
 * "a fold over the entire prefix" (§2) that the prefill "folds ... per
 * chunk" (§5).  The method (a chunked scan) reaches exactly this result up
 * to rounding order, so the oracle is the definition itself: strictly sequential in t,
 * no chunking, no blocking, no reordering.
 *
 * Per (b, h), with row vectors q_t, k_t in R^{dk}, v_t in R^{dv}, scalar g_t in (0,1]:
 *     S_0 = state_in                        (dk x dv)
 *     S_t = g_t * S_{t-1} + k_t^T v_t       (outer product)
 *     o_t = q_t S_t                         (uses the post-update state, s <= t inclusive)
 *     state_out = S_T
 *
 * Inputs q, k, v, g are float arrays that hold the already-rounded bf16 / fp32 input
 * values (widened exactly); every arithmetic operation below is in double.
 *
 * Layouts (row-major, contiguous innermost):
 *     q, k : [B, t_stride, H, dk]   (only tokens [0,T) of each batch are read)
 *     v    : [B, t_stride, H, dv]
 *     g    : [B, t_stride, H]
 *     state_in, state_out : [B, H, dk, dv]   (state_in may be NULL = zeros)
 *     o    : [B, T, H, dv]  (dense in T)
 *
 * Parallelism: OpenMP across (b, h) only — the t loop is never split.
 */
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int esc_oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* returns 0 on success, -1 on bad arguments, -2 on allocation failure */
int esc_oracle_linattn(const float* q, const float* k, const float* v, const float* g,
                       const double* state_in, double* o, double* state_out,
                       int64_t B, int64_t T, int64_t t_stride, int64_t H,
                       int64_t dk, int64_t dv, int n_threads) {
    if (!q || !k || !v || !g || !o || !state_out) return -1;
    if (B < 0 || T < 0 || H <= 0 || dk <= 0 || dv <= 0 || t_stride < T) return -1;
    int failed = 0;
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
#else
    (void)n_threads;
#endif
    const int64_t BH = B * H;
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
    for (int64_t bh = 0; bh < BH; ++bh) {
        const int64_t b = bh / H, h = bh % H;
        double* S = (double*)malloc((size_t)(dk * dv) * sizeof(double));
        if (!S) {
#pragma omp atomic write
            failed = 1;
            continue;
        }
        if (state_in)
            memcpy(S, state_in + (size_t)bh * dk * dv, (size_t)(dk * dv) * sizeof(double));
        else
            for (int64_t i = 0; i < dk * dv; ++i) S[i] = 0.0;

        for (int64_t t = 0; t < T; ++t) {
            const size_t tok = (size_t)(b * t_stride + t) * H + h;
            const float* qt = q + tok * dk;
            const float* kt = k + tok * dk;
            const float* vt = v + tok * dv;
            const double gt = (double)g[tok];
            double* ot = o + ((size_t)(b * T + t) * H + h) * dv;
            /* S_t = g_t S_{t-1} + k_t^T v_t */
            for (int64_t i = 0; i < dk; ++i) {
                const double ki = (double)kt[i];
                double* Si = S + i * dv;
                for (int64_t j = 0; j < dv; ++j) Si[j] = gt * Si[j] + ki * (double)vt[j];
            }
            /* o_t = q_t S_t */
            for (int64_t j = 0; j < dv; ++j) ot[j] = 0.0;
            for (int64_t i = 0; i < dk; ++i) {
                const double qi = (double)qt[i];
                const double* Si = S + i * dv;
                for (int64_t j = 0; j < dv; ++j) ot[j] += qi * Si[j];
            }
        }
        memcpy(state_out + (size_t)bh * dk * dv, S, (size_t)(dk * dv) * sizeof(double));
        free(S);
    }
    return failed ? -2 : 0;
}
