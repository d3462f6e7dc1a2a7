// Gated delta-rule scan, chunked (WY) form on the tensor cores with warp-level MMAs (include/esc.h: esc_gdn_scan).
//
//     u_t = k_t (a_t S_{t-1}) ,  S_t = a_t S_{t-1} + beta_t k_t^T (v_t - u_t) ,  o_t = q_t S_t
//
// Per chunk of 16 tokens, with S_0 the state at the chunk's start, b_i = sum_{r<=i} log2 a_r (inclusive, in the chunk),
// D_ij = 2^(b_i - b_j):
//     X_k = K S_0 , X_q = Q S_0                               (16 x d_v each)      mma  M = d_v slice, N = 16 tokens, K = d_k
//     G_kk = K K^T , G_qk = Q K^T                             (16 x 16 each)       mma  M = 16 tokens, N = 16 tokens, K = d_k
//     w_i = beta_i (v_i - 2^(b_i) X_k,i - sum_{j<i} D_ij G_kk,ij w_j)              sequential: rank-1 updates of the residual,
//                                                                                   two columns per round of shuffles
//     o_i = 2^(b_i) X_q,i + sum_{j<=i} D_ij G_qk,ij w_j                            mma  M = d_v slice, N = 16, K = 16
//     S_16 = 2^(b_15) S_0 + sum_j 2^(b_15 - b_j) k_j^T w_j                         mma  M = d_v slice, N = d_k, K = 16
// which is the recurrence above with the 16 updates of a chunk expanded (exact in exact arithmetic).
//
// Decomposition: the columns of S are independent, so one CTA owns (b, h, 16 columns of d_v).  S^T (16 x d_k) lives in the fp32
// accumulator registers of the MMAs for the whole call: it is the C operand of the state update and — re-read as an A
// operand, a register-local relabelling of the accumulator fragments — the left factor of X^T = S^T K^T; every product is
// computed transposed (d_v rows) for that reason.  fp32 factors (S, w, the decayed Gram entries) enter the bf16 MMAs as
// two-term splits (hi + lo); q, k are the bf16 inputs themselves.
// Nine warps, by what depends on what:
//   warps 0-3  the recurrence: each holds a quarter of d_k (of the rows of S), computes its part of X_k, X_q, exchanges the
//              partial sums through shared memory (one named barrier per chunk, summed in warp order by every reader: same
//              bits everywhere), solves the 16 x 16 system (redundantly: no second barrier) and updates its quarter of S;
//              warp 0 leaves W of the chunk in a shared-memory slot for the output warps;
//   warps 4-5  the Gram matrices, decays and their products L, M: functions of the inputs only, computed one 64-token block
//              ahead into shared memory, alternate chunks each;
//   warp 6     cp.async loader, two blocks ahead (three input buffers, padded rows: conflict-free fragment loads);
//   warps 7-8  the outputs, off the carry chain: o of eight tokens of each chunk from the partial X_q, W and M (named
//              full / empty barriers per chunk parity; the recurrence runs up to two chunks ahead of them).
// One CTA barrier per block of 64 tokens hands the buffers on.  Tokens beyond T are staged as k = q = v = 0, beta = 0, a = 1:
// they leave the state alone.
// Bound: the per-chunk dependency chain of the recurrence warps (~1900 cycles per 16 tokens: X 230, exchange 400, residual
// 140, solve 520, o 300, state update 180; r01 clock64 accounting), not HBM and not the tensor pipe: B H d_v / 16 = 128
// independent chains is all the parallelism the recurrence has at B = 1.  Tried (r01): a token order that gives a lane four
// consecutive tokens (4 rounds of shuffles instead of 8, swizzled rows against the bank conflicts it causes): slower, the
// solve is bound by its instruction count, not by the shuffle rounds; hoisting every shared-memory load of the chain above
// the MMAs: slower.
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
constexpr int kGmGW = 2;            // Gram warps (one block ahead; the chunks of a block alternate between them)
constexpr int kGmOW = 2;            // output warps: o of eight tokens of each chunk, one chunk behind the recurrence
constexpr int kGmWarps = kGmRW + kGmGW + 1 + kGmOW;   // + the cp.async loader (two blocks ahead)
constexpr int kGmThreads = 32 * kGmWarps;
constexpr int kGmNB = 3;            // staged input blocks

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
// named barriers: 1 = the recurrence warps' exchange; 2, 3 = "W of the chunk is in its slot" (per chunk parity: recurrence warp 0
// arrives, the output warps wait); 4, 5 = "slot and partial sums of that parity consumed" (output warps arrive, recurrence warps wait)
constexpr int kGmBarFull = 2, kGmBarEmpty = 4;

template <int DK>
struct GmSmem {
    static constexpr int KS = DK + 8;              // padded row (bf16 elements): fragment loads hit 32 distinct banks
    __nv_bfloat16 q[kGmNB][kGmTB][KS];
    __nv_bfloat16 k[kGmNB][kGmTB][KS];
    __nv_bfloat16 v[kGmNB][kGmTB][kGmDVT];
    float a[kGmNB][kGmTB];
    float beta[kGmNB][kGmTB];
    struct Chunk {                                 // what the Gram warp hands to the recurrence warp, per 16-token chunk
        float L[kGmC][kGmC + 1];                   // beta_j D_ij G_kk,ij (j < i, else 0), fp32
        uint32_t Mhi[kGmC][kGmC / 2 + 1];          // D_ij G_qk,ij (j <= i, else 0): packed bf16 pairs over j, hi and lo terms
        uint32_t Mlo[kGmC][kGmC / 2 + 1];
        float bl[kGmC];                            // inclusive cumulative log2 decay
    } ch[2][kGmTB / kGmC];
    float4 wslot[2][2][32];                        // per chunk parity: W^T of the chunk in accumulator layout (8 values per lane)
    float4 part[2][kGmRW][4][32];                  // per chunk parity and recurrence warp: partial X_k^T (groups 0, 1 = n-tiles) and X_q^T (2, 3)
};

template <int DK>
__global__ void __launch_bounds__(kGmThreads) esc_gdn_mma_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ k,
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

    const uint64_t n_blocks = (T + kGmTB - 1) / kGmTB;
    auto stage = [&](uint64_t blk, int buf) {   // tokens [blk*TB, ...) -> buffer buf; the rest of the last chunk as identity tokens
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
            gm_cp_async16(&sm.v[buf][i >> 1][(i & 1) * 8], v + tok * DV + dv0 + (i & 1) * 8);
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
            *reinterpret_cast<uint4*>(&sm.v[buf][i >> 1][(i & 1) * 8]) = make_uint4(0, 0, 0, 0);
        for (int i = n + lane; i < n_pad; i += 32) {
            sm.a[buf][i] = 1.f;
            sm.beta[buf][i] = 0.f;
        }
    };

    // ---- Gram warp: decays, G_kk, G_qk of one chunk -> ck (depends on the inputs only: runs one block ahead) ----
    auto gram_chunk = [&](int buf, int c0, typename GmSmem<DK>::Chunk& ck) {
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
                ck.L[i][j0] = lv[0];
                ck.L[i][j0 + 1] = lv[1];
                uint32_t lo;
                ck.Mhi[i][j0 >> 1] = gm_split(mv[0], mv[1], lo);
                ck.Mlo[i][j0 >> 1] = lo;
            }
        }
    };
    // ---- recurrence warp: one chunk of the carry chain ----
    uint32_t chunk_no = 0;   // running chunk count (the parity picks the partial-sum buffer)
    const uint32_t total_chunks = (uint32_t)((T + C - 1) / C);
    auto main_chunk = [&](int buf, int c0, const typename GmSmem<DK>::Chunk& ck) {
        const int par = (int)(chunk_no & 1);
        // the output warps are done with the partial sums and the W slot of chunk_no - 2
        if (chunk_no >= 2) gm_bar_sync(kGmBarEmpty + par, 32 * (kGmRW + kGmOW));
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
        // exchange: every recurrence warp needs the whole X_k (summed in warp order by every reader: the same bits everywhere);
        // the partial X_q are summed by the output warps
        {
            float4(*pb)[4][32] = sm.part[chunk_no & 1];
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                pb[rw][nt][lane] = make_float4(xk[nt][0] + xkl[nt][0], xk[nt][1] + xkl[nt][1], xk[nt][2] + xkl[nt][2], xk[nt][3] + xkl[nt][3]);
                pb[rw][2 + nt][lane] = make_float4(xq[nt][0] + xql[nt][0], xq[nt][1] + xql[nt][1], xq[nt][2] + xql[nt][2], xq[nt][3] + xql[nt][3]);
            }
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
        // ---- residual R^T = V^T - 2^(b) X_k^T in accumulator layout: r[nt][e] = (row gq, token 8nt + 2c + e), r[nt][2+e] = row gq + 8 ----
        float r[2][4], eb[2][2], bt[2][2];
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int j = 8 * nt + 2 * c + e;
                eb[nt][e] = gm_ex2(ck.bl[j]);
                bt[nt][e] = sm.beta[buf][c0 + j];
                r[nt][e] = __bfloat162float(sm.v[buf][c0 + j][gq]) - eb[nt][e] * xk[nt][e];
                r[nt][2 + e] = __bfloat162float(sm.v[buf][c0 + j][gq + 8]) - eb[nt][e] * xk[nt][2 + e];
            }
        }
        // ---- the 16 x 16 unit-triangular system, right-looking: r_j -= (beta_i L_ji) r_i for j > i, then w = beta r.  Column i
        // lives in the lanes with c = (i % 8) / 2: shuffles broadcast it inside each 4-lane group.  L is zero on and above
        // the diagonal, so the update can run over every column a lane holds. ----
#pragma unroll
        for (int pr = 0; pr < C / 2; ++pr) {
            // columns i0 = 2 pr and i0 + 1 sit in the same lanes (c = pr % 4): the owner finishes column i0 + 1 itself, then both
            // columns are broadcast in one round of shuffles: 8 dependent rounds instead of 16
            const int i0c = 2 * pr, nti = pr >> 2, ci = pr & 3;
            const float l10 = ck.L[i0c + 1][i0c];
            const float a0 = r[nti][0], a1 = r[nti][2];
            const float b0 = fmaf(-l10, a0, r[nti][1]), b1 = fmaf(-l10, a1, r[nti][3]);
            const int src = (lane & ~3) | ci;
            const float wa0 = __shfl_sync(0xffffffffu, a0, src), wa1 = __shfl_sync(0xffffffffu, a1, src);
            const float wb0 = __shfl_sync(0xffffffffu, b0, src), wb1 = __shfl_sync(0xffffffffu, b1, src);
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                if (8 * nt + 7 <= i0c) continue;   // every column of this n-tile is <= i0: nothing below the diagonal
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int j = 8 * nt + 2 * c + e;
                    const float lja = ck.L[j][i0c], ljb = ck.L[j][i0c + 1];   // zero on and above the diagonal
                    r[nt][e] = fmaf(-ljb, wb0, fmaf(-lja, wa0, r[nt][e]));
                    r[nt][2 + e] = fmaf(-ljb, wb1, fmaf(-lja, wa1, r[nt][2 + e]));
                }
            }
        }
        float w[2][4];
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                w[nt][e] = bt[nt][e] * r[nt][e];
                w[nt][2 + e] = bt[nt][e] * r[nt][2 + e];
            }
        }
        // ---- hand W^T to the output warps (every recurrence warp holds the same W: warp 0 writes it) ----
        if (rw == 0) {
            sm.wslot[par][0][lane] = make_float4(w[0][0], w[0][1], w[0][2], w[0][3]);
            sm.wslot[par][1][lane] = make_float4(w[1][0], w[1][1], w[1][2], w[1][3]);
            gm_bar_arrive(kGmBarFull + par, 32 * (1 + kGmOW));
        }
        // ---- S^T <- 2^(b_15) S^T + (2^(b_15 - b_j) w_j)^T K  (B fragments of K by transposing ldmatrix) ----
        {
            const float blast = ck.bl[C - 1], gam = gm_ex2(blast);
            uint32_t wh[4], wl[4];
            float ws[2][4];
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const float sc = gm_ex2(blast - ck.bl[8 * nt + 2 * c + e]);
                    ws[nt][e] = sc * w[nt][e];
                    ws[nt][2 + e] = sc * w[nt][2 + e];
                }
            }
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
        ++chunk_no;
    };
    // ---- output warp ow: o of tokens 8 ow .. 8 ow + 7 of the chunk:  o^T = 2^(b) X_q^T + W^T M^T ----
    auto out_chunk = [&](int buf, int c0, const typename GmSmem<DK>::Chunk& ck, uint64_t t0, int n, int nt) {
        const int par = (int)(chunk_no & 1);
        gm_bar_sync(kGmBarFull + par, 32 * (1 + kGmOW));
        const float4 w0 = sm.wslot[par][0][lane], w1 = sm.wslot[par][1][lane];
        float4 sq = sm.part[par][0][2 + nt][lane];
#pragma unroll
        for (int w2 = 1; w2 < kGmRW; ++w2) {
            const float4 t = sm.part[par][w2][2 + nt][lane];
            sq.x += t.x; sq.y += t.y; sq.z += t.z; sq.w += t.w;
        }
        if (chunk_no + 2 < total_chunks) gm_bar_arrive(kGmBarEmpty + par, 32 * (kGmRW + kGmOW));   // slot and partial sums read
        const float xq[4] = {sq.x, sq.y, sq.z, sq.w};
        uint32_t wh[4], wl[4];
        wh[0] = gm_split(w0.x, w0.y, wl[0]);
        wh[1] = gm_split(w0.z, w0.w, wl[1]);
        wh[2] = gm_split(w1.x, w1.y, wl[2]);
        wh[3] = gm_split(w1.z, w1.w, wl[3]);
        const uint32_t mh0 = ck.Mhi[8 * nt + gq][c], mh1 = ck.Mhi[8 * nt + gq][4 + c];
        const uint32_t ml0 = ck.Mlo[8 * nt + gq][c], ml1 = ck.Mlo[8 * nt + gq][4 + c];
        float oa[4] = {0.f, 0.f, 0.f, 0.f}, ob[4] = {0.f, 0.f, 0.f, 0.f}, oc[4] = {0.f, 0.f, 0.f, 0.f};
        gm_mma(oa, wh, mh0, mh1);
        gm_mma(ob, wl, mh0, mh1);
        gm_mma(oc, wh, ml0, ml1);
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int j = 8 * nt + 2 * c + e;
            if (c0 + j < n) {
                const float ebj = gm_ex2(ck.bl[j]);
                float* op = o + (((size_t)b * t_stride + t0 + c0 + j) * H + h) * DV + dv0;
                op[gq] = fmaf(ebj, xq[e], oa[e] + (ob[e] + oc[e]));
                op[gq + 8] = fmaf(ebj, xq[2 + e], oa[2 + e] + (ob[2 + e] + oc[2 + e]));
            }
        }
        ++chunk_no;
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
        for (int c0 = gw * C; c0 < n0; c0 += kGmGW * C) gram_chunk(0, c0, sm.ch[0][c0 / C]);
    }
    __syncthreads();
    for (uint64_t blk = 0; blk < n_blocks; ++blk) {
        const uint64_t t0 = blk * kGmTB;
        const int n = (int)((T - t0) < (uint64_t)kGmTB ? (T - t0) : (uint64_t)kGmTB);
        if (warp < kGmRW) {
            for (int c0 = 0; c0 < n; c0 += C) main_chunk((int)(blk % kGmNB), c0, sm.ch[blk & 1][c0 / C]);
        } else if (warp > kGmRW + kGmGW) {
            for (int c0 = 0; c0 < n; c0 += C)
                out_chunk((int)(blk % kGmNB), c0, sm.ch[blk & 1][c0 / C], t0, n, warp - (kGmRW + kGmGW + 1));
        } else if (gw < kGmGW) {
            if (blk + 1 < n_blocks) {
                const uint64_t t1 = t0 + kGmTB;
                const int n1 = (int)((T - t1) < (uint64_t)kGmTB ? (T - t1) : (uint64_t)kGmTB);
                for (int c0 = gw * C; c0 < n1; c0 += kGmGW * C) gram_chunk((int)((blk + 1) % kGmNB), c0, sm.ch[(blk + 1) & 1][c0 / C]);
            }
        } else {
            if (blk + 2 < n_blocks) {
                stage(blk + 2, (int)((blk + 2) % kGmNB));
                gm_cp_wait<0>();
            }
        }
        __syncthreads();
    }
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
static int launch_gdn_mma_t(const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* beta,
                            const float* state_in, float* state_out, float* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    static bool attr_set = false;
    if (!attr_set) {
        ESC_CUDA(cudaFuncSetAttribute(esc_gdn_mma_kernel<DK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GmSmem<DK>)));
        attr_set = true;
    }
    dim3 grid(s.dv / kGmDVT, s.B * s.H);
    esc_gdn_mma_kernel<DK><<<grid, kGmThreads, sizeof(GmSmem<DK>), stream>>>(
        (const __nv_bfloat16*)q, (const __nv_bfloat16*)k, (const __nv_bfloat16*)v, g, beta, state_in, state_out, o, s.H, s.dv, T, t_stride);
    ESC_CUDA(cudaGetLastError());
    return ESC_OK;
}

int launch_gdn_mma(const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* beta,
                   const float* state_in, float* state_out, float* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    if (s.dv % kGmDVT) return ESC_ERR_UNSUPPORTED;
    if (s.dk == 128) return launch_gdn_mma_t<128>(s, q, k, v, g, beta, state_in, state_out, o, T, t_stride, stream);
    if (s.dk == 64) return launch_gdn_mma_t<64>(s, q, k, v, g, beta, state_in, state_out, o, T, t_stride, stream);
    return ESC_ERR_UNSUPPORTED;
}

}  // namespace esc
