// Gated delta-rule scan, chunked (WY) form on the tensor cores with warp-level MMAs (include/esc.h: esc_gdn_scan).
//
//     u_t = k_t (a_t S_{t-1}) ,  S_t = a_t S_{t-1} + beta_t k_t^T (v_t - u_t) ,  o_t = q_t S_t
//
// Per chunk of 16 tokens, with S_0 the state at the chunk's start, b_i = sum_{r<=i} log2 a_r (inclusive, in the chunk),
// D_ij = 2^(b_i - b_j), the 16 updates of a chunk expanded (exact in exact arithmetic; the chunked "WY" form):
//     X_k = K S_0 , X_q = Q S_0                               (16 x d_v each)      mma  M = d_v slice, N = 16 tokens, K = d_k
//     G_kk = K K^T , G_qk = Q K^T                             (16 x 16 each)       mma  M = 16 tokens, N = 16 tokens, K = d_k
//     L_ij = beta_j D_ij G_kk,ij (j < i) , M_ij = D_ij G_qk,ij (j <= i)
//     w_i = beta_i r_i ,  (I + L) r = R ,  R = V - diag(2^b) X_k                   the 16 x 16 unit-triangular system
//     o_i = 2^(b_i) X_q,i + sum_{j<=i} M_ij w_j                                    mma  M = d_v slice, N = 16, K = 16
//     S_16 = 2^(b_15) S_0 + sum_j 2^(b_15 - b_j) k_j^T w_j                         mma  M = d_v slice, N = d_k, K = 16
// The system is not solved on the carry chain: N = diag(beta) (I + L)^-1 depends on k, beta, a only, so it is formed ahead of
// the chain (forward substitution, one column per lane), and with U = diag(2^(b_15 - b)) N, E = -U diag(2^b) the decayed W the
// state update takes is one small product with what the chain has just computed:
//     diag(2^(b_15 - b)) W = U R = U V + E X_k                                     mma  M = d_v slice, N = 16, K = 16
// (U V, a function of the inputs, is also formed ahead); the outputs take W = N R off the chain.
//
// Decomposition: the columns of S are independent, so one CTA owns (b, h, 16 columns of d_v).  S^T (16 x d_k) lives in the fp32
// accumulator registers of the MMAs for the whole call: it is the C operand of the state update and — re-read as an A
// operand, a register-local relabelling of the accumulator fragments — the left factor of X^T = S^T K^T; every product is
// computed transposed (d_v rows) for that reason.  fp32 factors (S, X_k, R, W, N, U, E, M) enter the bf16 MMAs as two-term
// splits (hi + lo; hi hi + lo hi + hi lo where both factors are split); q, k, v are the bf16 inputs themselves.
// Eleven warps, by what depends on what:
//   warps 0-3  the recurrence (the carry chain): each holds a quarter of d_k (of the rows of S), computes its part of X_k, X_q,
//              exchanges the partial sums through shared memory (one named barrier per chunk, summed in warp order by every
//              reader: same bits everywhere), forms the decayed W (redundantly: no second barrier) and updates its quarter of S;
//   warps 4-7  one chunk of each 64-token block each, one block ahead: decays, Gram matrices, L, M, the inverse N, U, E and
//              U V into shared memory: functions of the inputs only;
//   warp 8     cp.async loader, two blocks ahead (three q / k buffers, padded rows: conflict-free fragment loads);
//   warps 9-10 the outputs, whole chunks in turn: R from the partial X_k, W = N R, o from the partial X_q, W and M.  They follow
//              the recurrence through named full / empty barriers per set of partial sums (four sets) and take no part in the
//              per-block barrier: v and the per-chunk products are kept one block longer than their producers need.
// One barrier of warps 0-8 per block of 64 tokens hands the buffers on.  Tokens beyond T are staged as k = q = v = 0,
// beta = 0, a = 1: they leave the state alone.
// Bound: the per-chunk dependency chain of the recurrence warps (~1450 cycles per 16 tokens, r01 clock64 accounting of the
// trace build -DESC_GM_PROF: S split + X MMAs ~330, exchange ~450, decayed W ~150, state update ~200, waits for the MMA
// results in between), not HBM and not the tensor pipe: B H d_v / 16 = 128 independent chains is all the parallelism the
// recurrence has at B = 1.  History (r01): the system solved on the chain by 8 rounds of shuffles (~520 cycles of ~1900) with
// two Gram warps: 1.02 ms at 16 448 tokens; o on warps of its own: 0.95 ms; the inverse ahead of the chain: 0.78 ms (it needs
// four Gram warps: 1.10 ms with two).  Tried and not faster: a token order that gives a lane four consecutive tokens for the
// solve; hoisting every shared-memory load of the chain above the MMAs; three output warps or two sets of partial sums.
//
// Restore + continue is bit-identical to the cold run when the boundary is a multiple of 16 tokens from the start of the
// sequence of calls (every chunk-aligned boundary is); elsewhere it agrees to rounding.
#include <cuda_bf16.h>

#include "esc_internal.h"

namespace esc {

constexpr int kGmTB = 64;          // tokens per staged block
constexpr int kGmC = 16;           // tokens per chunk
constexpr int kGmDVT = 16;         // d_v columns per warp / CTA
constexpr int kGmRW = 4;            // recurrence warps: each owns a quarter of d_k (of the rows of S)
#ifndef ESC_GM_GW
#define ESC_GM_GW 4
#endif
constexpr int kGmGW = ESC_GM_GW;            // Gram warps (one block ahead; the chunks of a block alternate between them)
#ifndef ESC_GM_OW
#define ESC_GM_OW 2
#endif
constexpr int kGmOW = ESC_GM_OW;    // output warps: whole chunks in turn (chunk n is warp n % kGmOW's), behind the recurrence
#ifndef ESC_GM_NP
#define ESC_GM_NP 4
#endif
constexpr int kGmNP = ESC_GM_NP;    // sets of partial sums in flight between the recurrence and the output warps
constexpr int kGmWarps = kGmRW + kGmGW + 1 + kGmOW;   // + the cp.async loader (two blocks ahead)
constexpr int kGmThreads = 32 * kGmWarps;
constexpr int kGmNB = 3;            // staged input blocks (q, k, a, beta)
constexpr int kGmNV = 4;            // staged v blocks, kGmNCH sets of per-chunk products: one more than their producers need, so that the
constexpr int kGmNCH = 3;           // output warps (up to two chunks behind the recurrence) stay out of the per-block barrier

__device__ __forceinline__ void gm_cp_async16(void* smem, const void* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void gm_cp_async4(void* smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void gm_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void gm_cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// D (16x8, fp32) += A (16x16, bf16, row) * B (16x8, bf16, col)
__device__ __forceinline__ void gm_mma(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t gm_pack(float x0, float x1) {   // element 0 in the low half
    __nv_bfloat162 p = __floats2bfloat162_rn(x0, x1);
    return *reinterpret_cast<uint32_t*>(&p);
}
// two-term split of a pair: packed hi terms returned, packed lo terms written
__device__ __forceinline__ uint32_t gm_split(float x0, float x1, uint32_t& lo) {
    const uint32_t hi = gm_pack(x0, x1);
    lo = gm_pack(x0 - __uint_as_float(hi << 16), x1 - __uint_as_float(hi & 0xFFFF0000u));
    return hi;
}
__device__ __forceinline__ float gm_ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// four 8x8 b16 matrices, transposed on the way: the B fragments (k = rows of smem, n = 8 consecutive columns) of two n-tiles
__device__ __forceinline__ void gm_ldmatrix_x4_trans(uint32_t (&r)[4], const void* row_ptr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"((uint32_t)__cvta_generic_to_shared(row_ptr)));
}

__device__ __forceinline__ void gm_bar_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void gm_bar_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }
// named barriers: 1 = the recurrence warps' exchange; kGmBarFull + p = "the partial sums of a chunk are in set p" (the recurrence
// warps arrive, the chunk's output warp waits); kGmBarEmpty + p = "that output warp has read all it needs of the chunk from shared
// memory" (it arrives, the recurrence warps wait before they write set p again); kGmBarBlock = the per-block barrier of every warp
// but the output warps
constexpr int kGmBarFull = 2, kGmBarEmpty = kGmBarFull + kGmNP, kGmBarBlock = kGmBarEmpty + kGmNP;
static_assert(kGmBarBlock <= 15, "named barriers");

#ifdef ESC_GM_PROF
// r01 cycle accounting (trace build only): [0..7] recurrence warp 0 of CTA (0, 0), [8..15] Gram warp 0, [16..23] output warp 0
__device__ long long g_gm_prof[24];
#define GM_STAMP(slot)                                                        \
    do {                                                                      \
        if (prof_on) {                                                        \
            const long long now_ = clock64();                                 \
            prof_acc[slot] += now_ - prof_t;                                  \
            prof_t = now_;                                                    \
        }                                                                     \
    } while (0)
#else
#define GM_STAMP(slot) do {} while (0)
#endif

template <int DK>
struct GmSmem {
    static constexpr int KS = DK + 8;              // padded row (bf16 elements): fragment loads hit 32 distinct banks
    __nv_bfloat16 q[kGmNB][kGmTB][KS];
    __nv_bfloat16 k[kGmNB][kGmTB][KS];
    __nv_bfloat16 v[kGmNV][kGmTB][kGmDVT];
    float a[kGmNB][kGmTB];
    float beta[kGmNB][kGmTB];
    struct Chunk {                                 // what the Gram warp hands to the recurrence warp, per 16-token chunk
        float LT[kGmC][kGmC + 4];                  // LT[j][i] = beta_j D_ij G_kk,ij (j < i, else 0), fp32: the Gram warp's own scratch
        uint32_t Mhi[kGmC][kGmC / 2 + 1];          // D_ij G_qk,ij (j <= i, else 0): packed bf16 pairs over j, hi and lo terms
        uint32_t Mlo[kGmC][kGmC / 2 + 1];
        uint32_t Nhi[kGmC][kGmC / 2 + 1];          // N_ij = beta_i ((I + L)^-1)_ij: W = N R (the output warps), same packing
        uint32_t Nlo[kGmC][kGmC / 2 + 1];
        uint32_t Ehi[kGmC][kGmC / 2 + 1];          // E_ij = -2^(b_j) U_ij, U_ij = 2^(b_15 - b_i) N_ij: the decayed W the state update
        uint32_t Elo[kGmC][kGmC / 2 + 1];          // takes is U R = U V + E X_k
        float4 VU[2][32];                          // (U V)^T for this CTA's d_v slice, accumulator layout per n-tile
        float bl[kGmC];                            // inclusive cumulative log2 decay
    } ch[kGmNCH][kGmTB / kGmC];
    float4 part[kGmNP][kGmRW][4][32];                  // per chunk parity and recurrence warp: partial X_k^T (groups 0, 1 = n-tiles) and X_q^T (2, 3)
};

template <int DK>
__global__ void __launch_bounds__(kGmThreads, 1) esc_gdn_mma_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ k,
                                                                 const __nv_bfloat16* __restrict__ v, const float* __restrict__ g,
                                                                 const float* __restrict__ beta, const float* state_in, float* state_out,
                                                                 float* __restrict__ o, uint32_t H, uint32_t DV, uint64_t T,
                                                                 uint64_t t_stride) {
    extern __shared__ __align__(16) uint8_t gm_raw[];
    GmSmem<DK>& sm = *reinterpret_cast<GmSmem<DK>*>(gm_raw);
    static_assert(DK == 64 || DK == 128, "d_k");
    constexpr int NKS = DK / 16, NT = DK / 8, C = kGmC;
    constexpr int KPW = NKS / kGmRW, NTW = NT / kGmRW;   // k-steps / n-tiles of d_k per recurrence warp
    static_assert(KPW >= 1 && NTW == 2 * KPW, "d_k split");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, gq = lane >> 2, c = lane & 3;
    const uint32_t bh = blockIdx.y, b = bh / H, h = bh % H, dv0 = blockIdx.x * kGmDVT;

    // S^T (16 d_v rows x d_k) in accumulator layout, the d_k range [rw DK/4, (rw+1) DK/4) of it in recurrence warp rw:
    // St[l][0,1] = (row gq, d_k 8 (rw NTW + l) + 2c + {0,1}), St[l][2,3] = (row gq + 8, same)
    const int rw = warp < kGmRW ? warp : 0;
    float St[NTW][4];
#pragma unroll
    for (int l = 0; l < NTW; ++l) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const size_t dk = 8 * (rw * NTW + l) + 2 * c + (e & 1), dv = dv0 + gq + 8 * (e >> 1);
            St[l][e] = (warp < kGmRW && state_in) ? state_in[((size_t)bh * DK + dk) * DV + dv] : 0.f;
        }
    }

#ifdef ESC_GM_PROF
    const bool prof_on = blockIdx.x == 0 && blockIdx.y == 0 && lane == 0 && (warp == 0 || warp == kGmRW || warp == kGmRW + kGmGW + 1);
    long long prof_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, prof_t = clock64();
#endif
    const uint64_t n_blocks = (T + kGmTB - 1) / kGmTB;
    auto stage = [&](uint64_t blk, int buf) {
        const int vb = (int)(blk % kGmNV);   // tokens [blk*TB, ...) -> buffer buf; the rest of the last chunk as identity tokens
        const uint64_t t0 = blk * kGmTB;
        const int n = (int)((T - t0) < (uint64_t)kGmTB ? (T - t0) : (uint64_t)kGmTB);
        constexpr int CHK = DK / 8;                     // 16-byte pieces per token row of q / k
        for (int i = lane; i < n * CHK; i += 32) {
            const int tt = i / CHK, cc = i % CHK;
            const size_t tok = ((size_t)b * t_stride + t0 + tt) * H + h;
            gm_cp_async16(&sm.q[buf][tt][cc * 8], q + tok * DK + cc * 8);
            gm_cp_async16(&sm.k[buf][tt][cc * 8], k + tok * DK + cc * 8);
        }
        for (int i = lane; i < n * 2; i += 32) {
            const size_t tok = ((size_t)b * t_stride + t0 + (i >> 1)) * H + h;
            gm_cp_async16(&sm.v[vb][i >> 1][(i & 1) * 8], v + tok * DV + dv0 + (i & 1) * 8);
        }
        for (int i = lane; i < n; i += 32) {
            const size_t tok = ((size_t)b * t_stride + t0 + i) * H + h;
            gm_cp_async4(&sm.a[buf][i], g + tok);
            gm_cp_async4(&sm.beta[buf][i], beta + tok);
        }
        gm_cp_commit();
        const int n_pad = (n + C - 1) / C * C;
        for (int i = n * CHK + lane; i < n_pad * CHK; i += 32) {
            const int tt = i / CHK, cc = i % CHK;
            *reinterpret_cast<uint4*>(&sm.q[buf][tt][cc * 8]) = make_uint4(0, 0, 0, 0);
            *reinterpret_cast<uint4*>(&sm.k[buf][tt][cc * 8]) = make_uint4(0, 0, 0, 0);
        }
        for (int i = n * 2 + lane; i < n_pad * 2; i += 32)
            *reinterpret_cast<uint4*>(&sm.v[vb][i >> 1][(i & 1) * 8]) = make_uint4(0, 0, 0, 0);
        for (int i = n + lane; i < n_pad; i += 32) {
            sm.a[buf][i] = 1.f;
            sm.beta[buf][i] = 0.f;
        }
    };

    // ---- Gram warp: decays, G_kk, G_qk of one chunk -> ck (depends on the inputs only: runs one block ahead) ----
    auto gram_chunk = [&](int buf, int vb, int c0, typename GmSmem<DK>::Chunk& ck) {
        GM_STAMP(0);
        {   // bl[i] = sum_{r<=i} log2 a_r (warp scan over lanes 0..15, fixed order)
            float lg = lane < C ? log2f(sm.a[buf][c0 + lane]) : 0.f;
#pragma unroll
            for (int d = 1; d < C; d <<= 1) {
                const float up = __shfl_up_sync(0xffffffffu, lg, d);
                if (lane >= d) lg += up;
            }
            if (lane < C) ck.bl[lane] = lg;
            __syncwarp();
        }
        float gkk[2][4] = {}, gqk[2][4] = {};
#pragma unroll
        for (int ks = 0; ks < NKS; ++ks) {
            uint32_t bk[2][2], aq[4];
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                const __nv_bfloat16* kr = &sm.k[buf][c0 + 8 * nt + gq][16 * ks + 2 * c];
                const __nv_bfloat16* qr = &sm.q[buf][c0 + 8 * nt + gq][16 * ks + 2 * c];
                bk[nt][0] = *reinterpret_cast<const uint32_t*>(kr);
                bk[nt][1] = *reinterpret_cast<const uint32_t*>(kr + 8);
                aq[nt] = *reinterpret_cast<const uint32_t*>(qr);          // A fragment: a0 / a1 = rows gq / gq + 8, k 2c ..
                aq[2 + nt] = *reinterpret_cast<const uint32_t*>(qr + 8);  //             a2 / a3 = the same rows, k 2c + 8 ..
            }
            // the K registers read as an A fragment (rows = tokens gq, gq + 8)
            const uint32_t ak[4] = {bk[0][0], bk[1][0], bk[0][1], bk[1][1]};
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                gm_mma(gkk[nt], ak, bk[nt][0], bk[nt][1]);
                gm_mma(gqk[nt], aq, bk[nt][0], bk[nt][1]);
            }
        }
        GM_STAMP(1);
        // decayed entries: L (fp32, strictly lower) and M (bf16 hi/lo pairs, lower incl. diagonal); zero elsewhere
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) {
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                const int i = gq + 8 * hf, j0 = 8 * nt + 2 * c;
                float lv[2], mv[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int j = j0 + e;
                    const float d = gm_ex2(ck.bl[i] - ck.bl[j]);
                    lv[e] = j < i ? d * gkk[nt][2 * hf + e] * sm.beta[buf][c0 + j] : 0.f;   // beta_j folded in: r_i -= L_ij r_j
                    mv[e] = j <= i ? d * gqk[nt][2 * hf + e] : 0.f;
                }
                ck.LT[j0][i] = lv[0];
                ck.LT[j0 + 1][i] = lv[1];
                uint32_t lo;
                ck.Mhi[i][j0 >> 1] = gm_split(mv[0], mv[1], lo);
                ck.Mlo[i][j0 >> 1] = lo;
            }
        }
        __syncwarp();
        GM_STAMP(2);
        // (I + L)^-1, column by column: lane col solves (I + L) x = e_col by forward substitution (fp32, fixed order; the columns of
        // L are warp-wide broadcast reads).  It depends on k, beta, a only, so it is off the carry chain; the chain then gets
        // W = N R with one small MMA instead of a 16-step solve.
        {
            const int col = lane & (C - 1);
            float x[C];
#pragma unroll
            for (int i = 0; i < C; ++i) x[i] = (i == col) ? 1.f : 0.f;
            // right-looking: once x_j is final, every later row takes its term (independent FMAs; the chain is one FMA per column)
#pragma unroll
            for (int j = 0; j + 1 < C; ++j) {
#pragma unroll
                for (int i4 = (j + 1) / 4; i4 < C / 4; ++i4) {
                    const float4 l4 = *reinterpret_cast<const float4*>(&ck.LT[j][4 * i4]);
                    if (4 * i4 + 0 > j) x[4 * i4 + 0] = fmaf(-l4.x, x[j], x[4 * i4 + 0]);
                    if (4 * i4 + 1 > j) x[4 * i4 + 1] = fmaf(-l4.y, x[j], x[4 * i4 + 1]);
                    if (4 * i4 + 2 > j) x[4 * i4 + 2] = fmaf(-l4.z, x[j], x[4 * i4 + 2]);
                    if (4 * i4 + 3 > j) x[4 * i4 + 3] = fmaf(-l4.w, x[j], x[4 * i4 + 3]);
                }
            }
            GM_STAMP(3);
            // lane col holds column col: through shared memory (the LT scratch, now consumed) into the (row, column pair)
            // ownership the packed operands are written in
            __syncwarp();
            if (lane < C) {
#pragma unroll
                for (int i = 0; i < C; ++i) ck.LT[i][col] = x[i];
            }
            __syncwarp();
            const float blast = ck.bl[C - 1];
            uint32_t uh[2][2], ul[2][2];   // [row half][column n-tile]: U as the B fragments of this very lane (rows 8 hf + gq)
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    const int i = gq + 8 * hf, j0 = 8 * nt + 2 * c;
                    const float2 nx = *reinterpret_cast<const float2*>(&ck.LT[i][j0]);
                    const float bi = sm.beta[buf][c0 + i], di = gm_ex2(blast - ck.bl[i]);
                    const float n0 = bi * nx.x, n1 = bi * nx.y, u0 = di * n0, u1 = di * n1;
                    uint32_t lo;
                    ck.Nhi[i][j0 >> 1] = gm_split(n0, n1, lo);
                    ck.Nlo[i][j0 >> 1] = lo;
                    uh[hf][nt] = gm_split(u0, u1, ul[hf][nt]);
                    ck.Ehi[i][j0 >> 1] = gm_split(-gm_ex2(ck.bl[j0]) * u0, -gm_ex2(ck.bl[j0 + 1]) * u1, lo);
                    ck.Elo[i][j0 >> 1] = lo;
                }
            }
            // (U V)^T = V^T U^T for the d_v slice (A = V^T by transposing ldmatrix: matrix m = lane / 8 is tokens 8 (m / 2) ..,
            // d_v 8 (m % 2) ..; B = U^T from the registers above; v is exact in bf16: two terms)
            uint32_t av[4];
            gm_ldmatrix_x4_trans(av, &sm.v[vb][c0 + (lane & 7) + 8 * (lane >> 4)][8 * ((lane >> 3) & 1)]);
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                float va[4] = {0.f, 0.f, 0.f, 0.f}, vb[4] = {0.f, 0.f, 0.f, 0.f};
                gm_mma(va, av, uh[nt][0], uh[nt][1]);
                gm_mma(vb, av, ul[nt][0], ul[nt][1]);
                ck.VU[nt][lane] = make_float4(va[0] + vb[0], va[1] + vb[1], va[2] + vb[2], va[3] + vb[3]);
            }
        }
        GM_STAMP(4);
    };
    // ---- recurrence warp: one chunk of the carry chain ----
    uint32_t chunk_no = 0;   // running chunk count (the parity picks the partial-sum buffer)
    const uint32_t total_chunks = (uint32_t)((T + C - 1) / C);
    auto main_chunk = [&](int buf, int c0, const typename GmSmem<DK>::Chunk& ck) {
        const int par = (int)(chunk_no % kGmNP);
        GM_STAMP(0);
        // partial X_k^T, X_q^T (d_v x tokens) over this warp's quarter of d_k; hi and lo terms of S accumulate separately
        float xk[2][4] = {}, xq[2][4] = {}, xkl[2][4] = {}, xql[2][4] = {};
#pragma unroll
        for (int kl = 0; kl < KPW; ++kl) {
            const int ks = rw * KPW + kl;
            uint32_t ah[4], al[4];
            ah[0] = gm_split(St[2 * kl][0], St[2 * kl][1], al[0]);
            ah[1] = gm_split(St[2 * kl][2], St[2 * kl][3], al[1]);
            ah[2] = gm_split(St[2 * kl + 1][0], St[2 * kl + 1][1], al[2]);
            ah[3] = gm_split(St[2 * kl + 1][2], St[2 * kl + 1][3], al[3]);
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                const __nv_bfloat16* kr = &sm.k[buf][c0 + 8 * nt + gq][16 * ks + 2 * c];
                const __nv_bfloat16* qr = &sm.q[buf][c0 + 8 * nt + gq][16 * ks + 2 * c];
                const uint32_t bk0 = *reinterpret_cast<const uint32_t*>(kr), bk1 = *reinterpret_cast<const uint32_t*>(kr + 8);
                const uint32_t bq0 = *reinterpret_cast<const uint32_t*>(qr), bq1 = *reinterpret_cast<const uint32_t*>(qr + 8);
                gm_mma(xk[nt], ah, bk0, bk1);
                gm_mma(xq[nt], ah, bq0, bq1);
                gm_mma(xkl[nt], al, bk0, bk1);
                gm_mma(xql[nt], al, bq0, bq1);
            }
        }
        GM_STAMP(2);
        // what the chain takes from the Gram warps, loaded ahead of the barrier
        const float4 vu0 = ck.VU[0][lane], vu1 = ck.VU[1][lane];
        uint32_t eh[2][2], el[2][2];
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) {
            eh[nt][0] = ck.Ehi[8 * nt + gq][c];
            eh[nt][1] = ck.Ehi[8 * nt + gq][4 + c];
            el[nt][0] = ck.Elo[8 * nt + gq][c];
            el[nt][1] = ck.Elo[8 * nt + gq][4 + c];
        }
        const float gam = gm_ex2(ck.bl[C - 1]);
        // exchange: every recurrence warp needs the whole X_k (summed in warp order by every reader: the same bits everywhere);
        // the output warps sum X_k and X_q for themselves
        {
            // the output warp of chunk_no - kGmNP is done with this set
            if (chunk_no >= (uint32_t)kGmNP) gm_bar_sync(kGmBarEmpty + par, 32 * (kGmRW + 1));
            GM_STAMP(1);
            float4(*pb)[4][32] = sm.part[par];
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                pb[rw][nt][lane] = make_float4(xk[nt][0] + xkl[nt][0], xk[nt][1] + xkl[nt][1], xk[nt][2] + xkl[nt][2], xk[nt][3] + xkl[nt][3]);
                pb[rw][2 + nt][lane] = make_float4(xq[nt][0] + xql[nt][0], xq[nt][1] + xql[nt][1], xq[nt][2] + xql[nt][2], xq[nt][3] + xql[nt][3]);
            }
            gm_bar_arrive(kGmBarFull + par, 32 * (kGmRW + 1));
            asm volatile("bar.sync 1, %0;" ::"n"(32 * kGmRW) : "memory");
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                float4 sk = pb[0][nt][lane];
#pragma unroll
                for (int w2 = 1; w2 < kGmRW; ++w2) {
                    const float4 t = pb[w2][nt][lane];
                    sk.x += t.x; sk.y += t.y; sk.z += t.z; sk.w += t.w;
                }
                xk[nt][0] = sk.x; xk[nt][1] = sk.y; xk[nt][2] = sk.z; xk[nt][3] = sk.w;
            }
        }
        GM_STAMP(3);
        // ---- the 16 x 16 unit-triangular system as products with its precomputed inverse: the decayed W^T the state update
        // takes, (2^(b_15 - b_j) w_j)^T = (U V)^T + X_k^T E^T  (A = X_k^T from the registers above, B from E in shared memory) ----
        float ws[2][4] = {{vu0.x, vu0.y, vu0.z, vu0.w}, {vu1.x, vu1.y, vu1.z, vu1.w}};
        {
            uint32_t xh[4], xl[4];
            xh[0] = gm_split(xk[0][0], xk[0][1], xl[0]);
            xh[1] = gm_split(xk[0][2], xk[0][3], xl[1]);
            xh[2] = gm_split(xk[1][0], xk[1][1], xl[2]);
            xh[3] = gm_split(xk[1][2], xk[1][3], xl[3]);
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                float wb[4] = {0.f, 0.f, 0.f, 0.f}, wc[4] = {0.f, 0.f, 0.f, 0.f};
                gm_mma(ws[nt], xh, eh[nt][0], eh[nt][1]);
                gm_mma(wb, xl, eh[nt][0], eh[nt][1]);
                gm_mma(wc, xh, el[nt][0], el[nt][1]);
#pragma unroll
                for (int e = 0; e < 4; ++e) ws[nt][e] += wb[e] + wc[e];
            }
        }
        GM_STAMP(5);
        // ---- S^T <- 2^(b_15) S^T + (2^(b_15 - b_j) w_j)^T K  (B fragments of K by transposing ldmatrix) ----
        {
            uint32_t wh[4], wl[4];
            wh[0] = gm_split(ws[0][0], ws[0][1], wl[0]);
            wh[1] = gm_split(ws[0][2], ws[0][3], wl[1]);
            wh[2] = gm_split(ws[1][0], ws[1][1], wl[2]);
            wh[3] = gm_split(ws[1][2], ws[1][3], wl[3]);
#pragma unroll
            for (int pl = 0; pl < NTW / 2; ++pl) {
                const int p = rw * (NTW / 2) + pl;
                uint32_t kb[4];
                // matrix m = lane / 8: rows = tokens 8 (m % 2) + lane % 8, columns = d_k 16 p + 8 (m / 2) ..
                gm_ldmatrix_x4_trans(kb, &sm.k[buf][c0 + 8 * ((lane >> 3) & 1) + (lane & 7)][16 * p + 8 * (lane >> 4)]);
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    St[2 * pl][e] *= gam;
                    St[2 * pl + 1][e] *= gam;
                }
                gm_mma(St[2 * pl], wh, kb[0], kb[1]);
                gm_mma(St[2 * pl + 1], wh, kb[2], kb[3]);
                gm_mma(St[2 * pl], wl, kb[0], kb[1]);
                gm_mma(St[2 * pl + 1], wl, kb[2], kb[3]);
            }
        }
        GM_STAMP(6);
        ++chunk_no;
    };
    // ---- output warp, one whole chunk:  R^T = V^T - 2^(b) X_k^T,  W^T = R^T N^T,  o^T = 2^(b) X_q^T + W^T M^T ----
    auto out_chunk = [&](int vb, int c0, const typename GmSmem<DK>::Chunk& ck, uint64_t t0, int n) {
        const int par = (int)(chunk_no % kGmNP);
        GM_STAMP(0);
        gm_bar_sync(kGmBarFull + par, 32 * (kGmRW + 1));
        GM_STAMP(1);
        float xk[2][4], xq[2][4];
#pragma unroll
        for (int n2 = 0; n2 < 2; ++n2) {
            float4 sk = sm.part[par][0][n2][lane], sq = sm.part[par][0][2 + n2][lane];
#pragma unroll
            for (int w2 = 1; w2 < kGmRW; ++w2) {
                const float4 t = sm.part[par][w2][n2][lane], u = sm.part[par][w2][2 + n2][lane];
                sk.x += t.x; sk.y += t.y; sk.z += t.z; sk.w += t.w;
                sq.x += u.x; sq.y += u.y; sq.z += u.z; sq.w += u.w;
            }
            xk[n2][0] = sk.x; xk[n2][1] = sk.y; xk[n2][2] = sk.z; xk[n2][3] = sk.w;
            xq[n2][0] = sq.x; xq[n2][1] = sq.y; xq[n2][2] = sq.z; xq[n2][3] = sq.w;
        }
        GM_STAMP(2);
        // residual in accumulator layout: r[n2][e] = (row gq, token 8 n2 + 2c + e), r[n2][2 + e] = row gq + 8
        float r[2][4], eb[2][2];
#pragma unroll
        for (int n2 = 0; n2 < 2; ++n2) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int j = 8 * n2 + 2 * c + e;
                eb[n2][e] = gm_ex2(ck.bl[j]);
                r[n2][e] = __bfloat162float(sm.v[vb][c0 + j][gq]) - eb[n2][e] * xk[n2][e];
                r[n2][2 + e] = __bfloat162float(sm.v[vb][c0 + j][gq + 8]) - eb[n2][e] * xk[n2][2 + e];
            }
        }
        // W^T = R^T N^T
        float w[2][4];
        {
            uint32_t rh[4], rl[4];
            rh[0] = gm_split(r[0][0], r[0][1], rl[0]);
            rh[1] = gm_split(r[0][2], r[0][3], rl[1]);
            rh[2] = gm_split(r[1][0], r[1][1], rl[2]);
            rh[3] = gm_split(r[1][2], r[1][3], rl[3]);
#pragma unroll
            for (int n2 = 0; n2 < 2; ++n2) {
                const uint32_t nh0 = ck.Nhi[8 * n2 + gq][c], nh1 = ck.Nhi[8 * n2 + gq][4 + c];
                const uint32_t nl0 = ck.Nlo[8 * n2 + gq][c], nl1 = ck.Nlo[8 * n2 + gq][4 + c];
                float wa[4] = {0.f, 0.f, 0.f, 0.f}, wb[4] = {0.f, 0.f, 0.f, 0.f}, wc[4] = {0.f, 0.f, 0.f, 0.f};
                gm_mma(wa, rh, nh0, nh1);
                gm_mma(wb, rl, nh0, nh1);
                gm_mma(wc, rh, nl0, nl1);
#pragma unroll
                for (int e = 0; e < 4; ++e) w[n2][e] = wa[e] + (wb[e] + wc[e]);
            }
        }
        uint32_t wh[4], wl[4];
        wh[0] = gm_split(w[0][0], w[0][1], wl[0]);
        wh[1] = gm_split(w[0][2], w[0][3], wl[1]);
        wh[2] = gm_split(w[1][0], w[1][1], wl[2]);
        wh[3] = gm_split(w[1][2], w[1][3], wl[3]);
        float oa[2][4] = {}, ob[2][4] = {}, oc[2][4] = {};
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) {
            const uint32_t mh0 = ck.Mhi[8 * nt + gq][c], mh1 = ck.Mhi[8 * nt + gq][4 + c];
            const uint32_t ml0 = ck.Mlo[8 * nt + gq][c], ml1 = ck.Mlo[8 * nt + gq][4 + c];
            gm_mma(oa[nt], wh, mh0, mh1);
            gm_mma(ob[nt], wl, mh0, mh1);
            gm_mma(oc[nt], wh, ml0, ml1);
        }
        // everything this chunk needs from shared memory is in registers
        if (chunk_no + kGmNP < total_chunks) gm_bar_arrive(kGmBarEmpty + par, 32 * (kGmRW + 1));
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int j = 8 * nt + 2 * c + e;
                if (c0 + j < n) {
                    float* op = o + (((size_t)b * t_stride + t0 + c0 + j) * H + h) * DV + dv0;
                    op[gq] = fmaf(eb[nt][e], xq[nt][e], oa[nt][e] + (ob[nt][e] + oc[nt][e]));
                    op[gq + 8] = fmaf(eb[nt][e], xq[nt][2 + e], oa[nt][2 + e] + (ob[nt][2 + e] + oc[nt][2 + e]));
                }
            }
        }
    };

    // ---- block pipeline: in period p the loader stages block p + 2, the Gram warp works on block p + 1, the recurrence on block p;
    // one CTA barrier per period (64 tokens) is all the synchronisation there is ----
    if (warp == kGmRW + kGmGW) {
        if (n_blocks > 0) stage(0, 0);
        if (n_blocks > 1) stage(1, 1);
        gm_cp_wait<0>();
    }
    __syncthreads();
    const int gw = warp - kGmRW;   // Gram warp index (valid for the Gram warps only)
    if (gw >= 0 && gw < kGmGW && n_blocks > 0) {
        const int n0 = (int)(T < (uint64_t)kGmTB ? T : (uint64_t)kGmTB);
        for (int c0 = gw * C; c0 < n0; c0 += kGmGW * C) gram_chunk(0, 0, c0, sm.ch[0][c0 / C]);
    }
    __syncthreads();
    for (uint64_t blk = 0; blk < n_blocks; ++blk) {
        const uint64_t t0 = blk * kGmTB;
        const int n = (int)((T - t0) < (uint64_t)kGmTB ? (T - t0) : (uint64_t)kGmTB);
        if (warp > kGmRW + kGmGW) {
            // the output warps follow the recurrence through the full / empty barriers alone: what they read of block blk (v,
            // the per-chunk products) is not overwritten before period blk + 2, and the recurrence enters period blk + 2 only
            // after its chunk 4 blk + 7 has waited for the output of chunk 4 blk + 7 - kGmNP >= 4 blk + 3 to be done with them
            static_assert(kGmNP <= kGmTB / kGmC, "output lag");
            const int ow = warp - (kGmRW + kGmGW + 1);
            for (int c0 = 0; c0 < n; c0 += C) {
                if ((int)(chunk_no % kGmOW) == ow) out_chunk((int)(blk % kGmNV), c0, sm.ch[blk % kGmNCH][c0 / C], t0, n);
                ++chunk_no;
            }
            continue;
        }
        if (warp < kGmRW) {
            for (int c0 = 0; c0 < n; c0 += C) main_chunk((int)(blk % kGmNB), c0, sm.ch[blk % kGmNCH][c0 / C]);
        } else if (gw < kGmGW) {
            if (blk + 1 < n_blocks) {
                const uint64_t t1 = t0 + kGmTB;
                const int n1 = (int)((T - t1) < (uint64_t)kGmTB ? (T - t1) : (uint64_t)kGmTB);
                for (int c0 = gw * C; c0 < n1; c0 += kGmGW * C)
                    gram_chunk((int)((blk + 1) % kGmNB), (int)((blk + 1) % kGmNV), c0, sm.ch[(blk + 1) % kGmNCH][c0 / C]);
            }
        } else {
            if (blk + 2 < n_blocks) {
                stage(blk + 2, (int)((blk + 2) % kGmNB));
                gm_cp_wait<0>();
            }
        }
        GM_STAMP(0);
        gm_bar_sync(kGmBarBlock, 32 * (kGmRW + kGmGW + 1));
        GM_STAMP(7);
    }
#ifdef ESC_GM_PROF
    if (prof_on)
        for (int i = 0; i < 8; ++i) g_gm_prof[(warp == 0 ? 0 : warp == kGmRW ? 8 : 16) + i] = prof_acc[i];
#endif
    if (warp >= kGmRW) return;
#pragma unroll
    for (int l = 0; l < NTW; ++l) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const size_t dk = 8 * (rw * NTW + l) + 2 * c + (e & 1), dv = dv0 + gq + 8 * (e >> 1);
            state_out[((size_t)bh * DK + dk) * DV + dv] = St[l][e];
        }
    }
}

template <int DK>
static int launch_gdn_mma_t(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* beta,
                            const float* state_in, float* state_out, float* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    const int rc = ensure_dyn_smem(ctx, kSlotGdn + (DK == 128 ? 0 : 1), esc_gdn_mma_kernel<DK>, (int)sizeof(GmSmem<DK>));
    if (rc != ESC_OK) return rc;
    dim3 grid(s.dv / kGmDVT, s.B * s.H);
    esc_gdn_mma_kernel<DK><<<grid, kGmThreads, sizeof(GmSmem<DK>), stream>>>(
        (const __nv_bfloat16*)q, (const __nv_bfloat16*)k, (const __nv_bfloat16*)v, g, beta, state_in, state_out, o, s.H, s.dv, T, t_stride);
    ESC_CUDA(cudaGetLastError());
    return ESC_OK;
}

#ifdef ESC_GM_PROF
extern "C" void esc_debug_gm_prof(long long* out24) { cudaMemcpyFromSymbol(out24, g_gm_prof, sizeof(g_gm_prof)); }
#endif

int launch_gdn_mma(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* beta,
                   const float* state_in, float* state_out, float* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    if (s.dv % kGmDVT) return ESC_ERR_UNSUPPORTED;
    if (s.dk == 128) return launch_gdn_mma_t<128>(ctx, s, q, k, v, g, beta, state_in, state_out, o, T, t_stride, stream);
    if (s.dk == 64) return launch_gdn_mma_t<64>(ctx, s, q, k, v, g, beta, state_in, state_out, o, T, t_stride, stream);
    return ESC_ERR_UNSUPPORTED;
}

}  // namespace esc
