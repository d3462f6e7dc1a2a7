/*
 * ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path (see linattn_oracle.c).
 *
 * (1) Gated delta-rule recurrence and (2) short causal depthwise convolution with a carried window — the two
 * folds of the paper's actual hybrid-model family: "the linear-attention recurrent state and convolution state
 * are a fold over the entire prefix [4, 13]" ([13] = Gated Delta Networks), both carried
 * by the capsule.  PAPER.md prints neither formula; reading 25 fixes them from [13]:
 *
 * (1) per (b, h), row vectors q_t, k_t in R^{dk}, v_t in R^{dv}, gate a_t in (0,1], write strength beta_t in [0,1]:
 *         u_t = k_t (a_t S_{t-1})                       (what the decayed memory returns for key k_t)
 *         S_t = a_t S_{t-1} + beta_t k_t^T (v_t - u_t)  ( = a_t (I - beta_t k_t^T k_t) S_{t-1} + beta_t k_t^T v_t )
 *         o_t = q_t S_t ,   state_out = S_T
 *     strictly sequential in t, fp64, OpenMP across (b, h) only.  Layouts as in linattn_oracle.c; beta like g.
 *
 * (2) per (b, channel c), window W, weights w[c][0..W):   y_t = sum_{i<W} w[c][i] * x_{t-W+1+i} , where x_s for s < 0
 *     is the carried state (the last W-1 inputs before the call, oldest first); optional SiLU y <- y / (1 + exp(-y));
 *     state_out = the last W-1 inputs after the call.  x: [B, t_stride, C]; w: [C, W]; state: [B, C, W-1]; y: [B, T, C].
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int esc_oracle_gdn(const float* q, const float* k, const float* v, const float* g, const float* beta,
                   const double* state_in, double* o, double* state_out,
                   int64_t B, int64_t T, int64_t t_stride, int64_t H, int64_t dk, int64_t dv, int n_threads) {
    if (!q || !k || !v || !g || !beta || !o || !state_out) return -1;
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
        double* S = (double*)malloc((size_t)(dk * dv + dv) * sizeof(double));
        if (!S) {
#pragma omp atomic write
            failed = 1;
            continue;
        }
        double* u = S + dk * dv;
        if (state_in) memcpy(S, state_in + (size_t)bh * dk * dv, (size_t)(dk * dv) * sizeof(double));
        else for (int64_t i = 0; i < dk * dv; ++i) S[i] = 0.0;
        for (int64_t t = 0; t < T; ++t) {
            const size_t tok = (size_t)(b * t_stride + t) * H + h;
            const float *qt = q + tok * dk, *kt = k + tok * dk, *vt = v + tok * dv;
            const double a = (double)g[tok], bt = (double)beta[tok];
            double* ot = o + ((size_t)(b * T + t) * H + h) * dv;
            /* decay, then u_t = k_t (a_t S_{t-1}) */
            for (int64_t i = 0; i < dk * dv; ++i) S[i] *= a;
            for (int64_t j = 0; j < dv; ++j) u[j] = 0.0;
            for (int64_t i = 0; i < dk; ++i)
                for (int64_t j = 0; j < dv; ++j) u[j] += (double)kt[i] * S[i * dv + j];
            /* S_t = a_t S_{t-1} + beta_t k_t^T (v_t - u_t) */
            for (int64_t i = 0; i < dk; ++i)
                for (int64_t j = 0; j < dv; ++j) S[i * dv + j] += bt * (double)kt[i] * ((double)vt[j] - u[j]);
            /* o_t = q_t S_t */
            for (int64_t j = 0; j < dv; ++j) ot[j] = 0.0;
            for (int64_t i = 0; i < dk; ++i)
                for (int64_t j = 0; j < dv; ++j) ot[j] += (double)qt[i] * S[i * dv + j];
        }
        memcpy(state_out + (size_t)bh * dk * dv, S, (size_t)(dk * dv) * sizeof(double));
        free(S);
    }
    return failed ? -2 : 0;
}

int esc_oracle_causal_conv(const float* x, const float* w, const double* state_in, double* y, double* state_out,
                           int64_t B, int64_t T, int64_t t_stride, int64_t C, int64_t W, int silu) {
    if (!x || !w || !y || !state_out || B < 0 || T < 0 || C <= 0 || W < 1 || t_stride < T) return -1;
    for (int64_t b = 0; b < B; ++b)
        for (int64_t c = 0; c < C; ++c) {
            for (int64_t t = 0; t < T; ++t) {
                double acc = 0.0;
                for (int64_t i = 0; i < W; ++i) {
                    const int64_t s = t - W + 1 + i;   /* input position of tap i */
                    double xs;
                    if (s >= 0) xs = (double)x[(size_t)(b * t_stride + s) * C + c];
                    else xs = state_in ? state_in[(size_t)(b * C + c) * (W - 1) + (W - 1 + s)] : 0.0;
                    acc += (double)w[c * W + i] * xs;
                }
                if (silu) acc = acc / (1.0 + exp(-acc));
                y[(size_t)(b * T + t) * C + c] = acc;
            }
            for (int64_t i = 0; i < W - 1; ++i) {      /* the last W-1 inputs, oldest first */
                const int64_t s = T - (W - 1) + i;
                double xs;
                if (s >= 0) xs = (double)x[(size_t)(b * t_stride + s) * C + c];
                else xs = state_in ? state_in[(size_t)(b * C + c) * (W - 1) + (W - 1 + s)] : 0.0;
                state_out[(size_t)(b * C + c) * (W - 1) + i] = xs;
            }
        }
    return 0;
}
