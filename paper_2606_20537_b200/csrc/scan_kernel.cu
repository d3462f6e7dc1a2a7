// Chunked gated linear-attention scan (include/esc.h: esc_linattn_scan).
//
// Definition (BASELINE.json north_star; "a fold over the entire prefix", folded
// "per chunk" PAPER.md:169):   S_t = g_t S_{t-1} + k_t^T v_t ,  o_t = q_t S_t.
// Chunk algebra evaluated here (exact-arithmetic equivalent; all exponents <= 0):
//     b_i    = sum_{r<=i in chunk} ln g_r
//     o_i    = exp(b_i) q_i S_prev + sum_{j<=i} exp(b_i - b_j) (q_i . k_j) v_j
//     S_next = exp(b_C) S_prev + sum_j exp(b_C - b_j) k_j^T v_j
//
// Decomposition: the columns of S (the d_v axis) are independent, so one CTA owns one
// (b, h, 32-column slice of d_v) and walks the chunks in order; the carry is a pure function
// of (S_prev bits, chunk inputs) — no T-dependent tiling, no atomics, no split-K — which is
// what makes restore-at-a-chunk-boundary + continue bit-identical to the cold run
// (PAPER.md:169-173).  The state slice lives in registers (fp32) for the whole scan.
//
// Precision plan (SURVEY.md §8(c) error budget): raw Q, K, V enter the tensor cores as the
// bf16 inputs they are; the three derived operands — A = (QK^T) ⊙ D, V~ = V ⊙ exp(b_C - b),
// S_prev — are split into two bf16 terms (hi + lo) and contracted with two MMAs into one
// fp32 accumulator, so every product carries >= 16 significand bits and stays range-safe.
// The row scale exp(b_i) of the inter-chunk term is applied in fp32 AFTER the contraction
// (Q S_prev is computed with the raw Q), so Q is never re-rounded.
//
// v0 tensor path: warp-level bf16 MMA (nvcuda::wmma, HMMA) with smem-staged operands.
#include <cuda_bf16.h>
#include <mma.h>

#include "esc_internal.h"

namespace esc {

using namespace nvcuda;
typedef __nv_bfloat16 bf16;

constexpr int kScanThreads = 256;
constexpr int kScanWarps = kScanThreads / 32;
constexpr int kDVT = 32;  // d_v columns per CTA

template <int DK, int C>
struct ScanSmem {
    static constexpr int LDQ = DK + 8;     // bf16 elements
    static constexpr int LDV = kDVT + 8;   // bf16
    static constexpr int LDA = C + 8;      // bf16
    static constexpr int LDP = C + 4;      // fp32
    static constexpr int LDO = kDVT + 4;   // fp32
    static constexpr int kStrip = 64;      // rows of P staged in fp32 at a time
    static constexpr size_t q_off = 0;
    static constexpr size_t k_off = q_off + (size_t)C * LDQ * 2;
    static constexpr size_t v_off = k_off + (size_t)C * LDQ * 2;
    static constexpr size_t vh_off = v_off + (size_t)C * LDV * 2;
    static constexpr size_t vl_off = vh_off + (size_t)C * LDV * 2;
    static constexpr size_t ah_off = vl_off + (size_t)C * LDV * 2;
    static constexpr size_t al_off = ah_off + (size_t)C * LDA * 2;
    static constexpr size_t sh_off = al_off + (size_t)C * LDA * 2;
    static constexpr size_t sl_off = sh_off + (size_t)DK * LDV * 2;
    static constexpr size_t scr_off = sl_off + (size_t)DK * LDV * 2;  // Pf strip | (Of, Uf)
    static constexpr size_t p_bytes = (size_t)kStrip * LDP * 4;
    static constexpr size_t o_bytes = (size_t)C * LDO * 4;
    static constexpr size_t u_bytes = (size_t)DK * LDO * 4;
    static constexpr size_t scr_bytes = p_bytes > o_bytes + u_bytes ? p_bytes : o_bytes + u_bytes;
    static constexpr size_t b_off = scr_off + scr_bytes;              // b[C], eb[C] fp32
    static constexpr size_t total = b_off + (size_t)2 * C * 4;
};

__device__ __forceinline__ void split_bf16(float x, bf16& hi, bf16& lo) {
    hi = __float2bfloat16_rn(x);
    lo = __float2bfloat16_rn(x - __bfloat162float(hi));
}

template <typename OutT>
__device__ __forceinline__ OutT to_out(float x);
template <>
__device__ __forceinline__ float to_out<float>(float x) { return x; }
template <>
__device__ __forceinline__ bf16 to_out<bf16>(float x) { return __float2bfloat16_rn(x); }

template <int DK, int C, typename OutT>
__global__ void __launch_bounds__(kScanThreads, 1)
esc_scan_kernel(const bf16* __restrict__ q, const bf16* __restrict__ k, const bf16* __restrict__ v,
                const float* __restrict__ g, const float* state_in, float* state_out, OutT* __restrict__ o,
                uint32_t H, uint32_t DV, uint64_t T, uint64_t t_stride) {
    using L = ScanSmem<DK, C>;
    extern __shared__ __align__(128) uint8_t smem[];
    bf16* Qs = (bf16*)(smem + L::q_off);
    bf16* Ks = (bf16*)(smem + L::k_off);
    bf16* Vs = (bf16*)(smem + L::v_off);
    bf16* Vh = (bf16*)(smem + L::vh_off);
    bf16* Vl = (bf16*)(smem + L::vl_off);
    bf16* Ah = (bf16*)(smem + L::ah_off);
    bf16* Al = (bf16*)(smem + L::al_off);
    bf16* Sh = (bf16*)(smem + L::sh_off);
    bf16* Sl = (bf16*)(smem + L::sl_off);
    float* Pf = (float*)(smem + L::scr_off);
    float* Of = (float*)(smem + L::scr_off);
    float* Uf = (float*)(smem + L::scr_off + L::o_bytes);
    float* bs = (float*)(smem + L::b_off);
    float* ebs = bs + C;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bh = blockIdx.y, b = bh / H, h = bh % H;
    const uint32_t dv0 = blockIdx.x * kDVT;

    // ---- state slice -> registers (+ hi/lo operand copy) ---------------------------------
    constexpr int kSReg = DK * kDVT / kScanThreads;
    float S[kSReg];
    {
        const size_t sbase = (size_t)bh * DK * DV + dv0;
#pragma unroll
        for (int r = 0; r < kSReg; ++r) {
            const int e = tid + r * kScanThreads, row = e / kDVT, col = e % kDVT;
            S[r] = state_in ? state_in[sbase + (size_t)row * DV + col] : 0.f;
            split_bf16(S[r], Sh[row * L::LDV + col], Sl[row * L::LDV + col]);
        }
    }

    const uint64_t n_chunks = (T + C - 1) / C;
    for (uint64_t c = 0; c < n_chunks; ++c) {
        const uint64_t t0 = c * C;
        const int n = (int)((T - t0) < (uint64_t)C ? (T - t0) : (uint64_t)C);
        const size_t tok0 = ((size_t)b * t_stride + t0) * H + h;  // token index of row 0 (x H stride per row)

        // ---- stage Q, K, V (bf16) and the cumulative log-decay -------------------------------
        {
            constexpr int VQ = DK / 8;  // 16-byte vectors per row
            for (int i = tid; i < C * VQ; i += kScanThreads) {
                const int row = i / VQ, vc = i % VQ;
                uint4 qv = make_uint4(0, 0, 0, 0), kv = qv;
                if (row < n) {
                    const size_t off = (tok0 + (size_t)row * H) * DK + vc * 8;
                    qv = *(const uint4*)(q + off);
                    kv = *(const uint4*)(k + off);
                }
                *(uint4*)(Qs + row * L::LDQ + vc * 8) = qv;
                *(uint4*)(Ks + row * L::LDQ + vc * 8) = kv;
            }
            constexpr int VV = kDVT / 8;
            for (int i = tid; i < C * VV; i += kScanThreads) {
                const int row = i / VV, vc = i % VV;
                uint4 vv = make_uint4(0, 0, 0, 0);
                if (row < n) vv = *(const uint4*)(v + (tok0 + (size_t)row * H) * DV + dv0 + vc * 8);
                *(uint4*)(Vs + row * L::LDV + vc * 8) = vv;
            }
            if (warp == 0) {  // b_i = inclusive prefix sum of ln g (warp shuffle scan, C/32 per lane)
                constexpr int PER = C / 32;
                float loc[PER];
                float run = 0.f;
#pragma unroll
                for (int u = 0; u < PER; ++u) {
                    const int i = lane * PER + u;
                    const float lg = i < n ? logf(g[tok0 + (size_t)i * H]) : 0.f;
                    run += lg;
                    loc[u] = run;
                }
                float incl = run;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const float up = __shfl_up_sync(0xffffffffu, incl, d);
                    if (lane >= d) incl += up;
                }
                const float excl = incl - run;
#pragma unroll
                for (int u = 0; u < PER; ++u) {
                    const float bi = excl + loc[u];
                    bs[lane * PER + u] = bi;
                    ebs[lane * PER + u] = __expf(bi);
                }
            }
        }
        __syncthreads();

        const float b_last = bs[C - 1];
        // ---- V~ = V ⊙ exp(b_C - b_j), two-term bf16 -------------------------------------------
        for (int i = tid; i < C * kDVT; i += kScanThreads) {
            const int row = i / kDVT, col = i % kDVT;
            const float x = __bfloat162float(Vs[row * L::LDV + col]) * __expf(b_last - bs[row]);
            split_bf16(x, Vh[row * L::LDV + col], Vl[row * L::LDV + col]);
        }

        // ---- A = (Q K^T) ⊙ D, lower-triangular tiles only, 64-row strips -----------------------
        for (int s0 = 0; s0 < C; s0 += L::kStrip) {
            {
                constexpr int TI = L::kStrip / 16, TJ = C / 16;
                for (int tix = warp; tix < TI * TJ; tix += kScanWarps) {
                    const int it = tix / TJ, jt = tix % TJ;
                    if (jt > it + s0 / 16) continue;
                    wmma::fragment<wmma::accumulator, 16, 16, 16, float> acc;
                    wmma::fill_fragment(acc, 0.f);
#pragma unroll
                    for (int kk = 0; kk < DK / 16; ++kk) {
                        wmma::fragment<wmma::matrix_a, 16, 16, 16, bf16, wmma::row_major> fa;
                        wmma::fragment<wmma::matrix_b, 16, 16, 16, bf16, wmma::col_major> fb;
                        wmma::load_matrix_sync(fa, Qs + (s0 + it * 16) * L::LDQ + kk * 16, L::LDQ);
                        wmma::load_matrix_sync(fb, Ks + (jt * 16) * L::LDQ + kk * 16, L::LDQ);
                        wmma::mma_sync(acc, fa, fb, acc);
                    }
                    wmma::store_matrix_sync(Pf + (it * 16) * L::LDP + jt * 16, acc, L::LDP, wmma::mem_row_major);
                }
            }
            __syncthreads();
            for (int i = tid; i < L::kStrip * C; i += kScanThreads) {
                const int rl = i / C, j = i % C, row = s0 + rl;
                if ((j >> 4) > (row >> 4)) continue;  // tile never read
                float a = 0.f;
                if (j <= row) a = Pf[rl * L::LDP + j] * __expf(bs[row] - bs[j]);
                split_bf16(a, Ah[row * L::LDA + j], Al[row * L::LDA + j]);
            }
            __syncthreads();
        }

        // ---- O = diag(exp b) (Q S_prev) + A V ;  U = K^T V~ ------------------------------------
        {
            constexpr int TI = C / 16, TN = kDVT / 16;
            for (int tix = warp; tix < TI * TN; tix += kScanWarps) {
                const int it = tix / TN, nt = tix % TN;
                wmma::fragment<wmma::accumulator, 16, 16, 16, float> acc;
                wmma::fill_fragment(acc, 0.f);
#pragma unroll
                for (int kk = 0; kk < DK / 16; ++kk) {
                    wmma::fragment<wmma::matrix_a, 16, 16, 16, bf16, wmma::row_major> fa;
                    wmma::fragment<wmma::matrix_b, 16, 16, 16, bf16, wmma::row_major> fh, fl;
                    wmma::load_matrix_sync(fa, Qs + (it * 16) * L::LDQ + kk * 16, L::LDQ);
                    wmma::load_matrix_sync(fh, Sh + (kk * 16) * L::LDV + nt * 16, L::LDV);
                    wmma::load_matrix_sync(fl, Sl + (kk * 16) * L::LDV + nt * 16, L::LDV);
                    wmma::mma_sync(acc, fa, fl, acc);
                    wmma::mma_sync(acc, fa, fh, acc);
                }
                // row scale exp(b_i) in fp32, through this warp's own smem tile
                float* ot = Of + (it * 16) * L::LDO + nt * 16;
                wmma::store_matrix_sync(ot, acc, L::LDO, wmma::mem_row_major);
                __syncwarp();
                for (int e = lane; e < 256; e += 32) {
                    const int r = e >> 4, cc = e & 15;
                    ot[r * L::LDO + cc] *= ebs[it * 16 + r];
                }
                __syncwarp();
                wmma::load_matrix_sync(acc, ot, L::LDO, wmma::mem_row_major);
                for (int kt = 0; kt <= it; ++kt) {
                    wmma::fragment<wmma::matrix_a, 16, 16, 16, bf16, wmma::row_major> fh, fl;
                    wmma::fragment<wmma::matrix_b, 16, 16, 16, bf16, wmma::row_major> fb;
                    wmma::load_matrix_sync(fh, Ah + (it * 16) * L::LDA + kt * 16, L::LDA);
                    wmma::load_matrix_sync(fl, Al + (it * 16) * L::LDA + kt * 16, L::LDA);
                    wmma::load_matrix_sync(fb, Vs + (kt * 16) * L::LDV + nt * 16, L::LDV);
                    wmma::mma_sync(acc, fl, fb, acc);
                    wmma::mma_sync(acc, fh, fb, acc);
                }
                wmma::store_matrix_sync(ot, acc, L::LDO, wmma::mem_row_major);
            }
            constexpr int TD = DK / 16;
            for (int tix = warp; tix < TD * TN; tix += kScanWarps) {
                const int dt = tix / TN, nt = tix % TN;
                wmma::fragment<wmma::accumulator, 16, 16, 16, float> acc;
                wmma::fill_fragment(acc, 0.f);
#pragma unroll
                for (int kt = 0; kt < C / 16; ++kt) {
                    wmma::fragment<wmma::matrix_a, 16, 16, 16, bf16, wmma::col_major> fa;  // K^T: (d, j) = Ks[j][d]
                    wmma::fragment<wmma::matrix_b, 16, 16, 16, bf16, wmma::row_major> fh, fl;
                    wmma::load_matrix_sync(fa, Ks + (kt * 16) * L::LDQ + dt * 16, L::LDQ);
                    wmma::load_matrix_sync(fh, Vh + (kt * 16) * L::LDV + nt * 16, L::LDV);
                    wmma::load_matrix_sync(fl, Vl + (kt * 16) * L::LDV + nt * 16, L::LDV);
                    wmma::mma_sync(acc, fa, fl, acc);
                    wmma::mma_sync(acc, fa, fh, acc);
                }
                wmma::store_matrix_sync(Uf + (dt * 16) * L::LDO + nt * 16, acc, L::LDO, wmma::mem_row_major);
            }
        }
        __syncthreads();

        // ---- write o ; carry S <- exp(b_C) S + U (fp32 registers) ; refresh S hi/lo -------------
        for (int i = tid; i < n * kDVT; i += kScanThreads) {
            const int row = i / kDVT, col = i % kDVT;
            o[(tok0 + (size_t)row * H) * DV + dv0 + col] = to_out<OutT>(Of[row * L::LDO + col]);
        }
        const float gam = __expf(b_last);
#pragma unroll
        for (int r = 0; r < kSReg; ++r) {
            const int e = tid + r * kScanThreads, row = e / kDVT, col = e % kDVT;
            S[r] = fmaf(gam, S[r], Uf[row * L::LDO + col]);
            split_bf16(S[r], Sh[row * L::LDV + col], Sl[row * L::LDV + col]);
        }
        __syncthreads();
    }

    {
        const size_t sbase = (size_t)bh * DK * DV + dv0;
#pragma unroll
        for (int r = 0; r < kSReg; ++r) {
            const int e = tid + r * kScanThreads, row = e / kDVT, col = e % kDVT;
            state_out[sbase + (size_t)row * DV + col] = S[r];
        }
    }
}

// ---- host ---------------------------------------------------------------------------------------
// key layout (opaque to callers): [63:56]=0xE5 tag, B:16, H:12, dk:8(/8), dv:8(/8), in:2, out:2, chunk:8(/8)
static const uint64_t kKeyTag = 0xE5ull;

bool decode_key(esc_shape_key key, ScanShape* s) {
    if ((key >> 56) != kKeyTag) return false;
    s->B = (uint32_t)((key >> 40) & 0xFFFF);
    s->H = (uint32_t)((key >> 28) & 0xFFF);
    s->dk = (uint32_t)((key >> 20) & 0xFF) * 8;
    s->dv = (uint32_t)((key >> 12) & 0xFF) * 8;
    s->in_dtype = (uint32_t)((key >> 10) & 3);
    s->out_dtype = (uint32_t)((key >> 8) & 3);
    s->chunk = (uint32_t)(key & 0xFF) * 8;
    return true;
}

template <int DK, int C, typename OutT>
static int launch_t(const ScanShape& s, const void* q, const void* k, const void* v, const float* g,
                    const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride,
                    cudaStream_t stream) {
    using L = ScanSmem<DK, C>;
    static bool attr_set = false;  // per-process, per-instantiation
    if (!attr_set) {
        ESC_CUDA(cudaFuncSetAttribute(esc_scan_kernel<DK, C, OutT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)L::total));
        attr_set = true;
    }
    if (!state_out) return ESC_OK;  // prepare-only call (before a stream capture)
    dim3 grid(s.dv / kDVT, s.B * s.H);
    esc_scan_kernel<DK, C, OutT><<<grid, kScanThreads, L::total, stream>>>(
        (const bf16*)q, (const bf16*)k, (const bf16*)v, g, state_in, state_out, (OutT*)o, s.H, s.dv, T, t_stride);
    ESC_CUDA(cudaGetLastError());
    return ESC_OK;
}

template <int DK, int C>
static int launch_o(const ScanShape& s, const void* q, const void* k, const void* v, const float* g,
                    const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride,
                    cudaStream_t stream) {
    if (s.out_dtype == ESC_DTYPE_F32)
        return launch_t<DK, C, float>(s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    return launch_t<DK, C, bf16>(s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
}

int launch_scan(const esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g,
                const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    (void)ctx;
    if (s.dk == 128 && s.chunk == 64) return launch_o<128, 64>(s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    if (s.dk == 128 && s.chunk == 128) return launch_o<128, 128>(s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    if (s.dk == 64 && s.chunk == 64) return launch_o<64, 64>(s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    if (s.dk == 64 && s.chunk == 128) return launch_o<64, 128>(s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    return ESC_ERR_UNSUPPORTED;
}

}  // namespace esc

using namespace esc;

extern "C" {

esc_shape_key esc_shape_key_make(uint32_t B, uint32_t H, uint32_t d_k, uint32_t d_v, uint32_t in_dtype,
                                 uint32_t out_dtype, uint32_t chunk) {
    if (B == 0 || H == 0 || B > 0xFFFF || H > 0xFFF || (uint64_t)B * H > 65535) return 0;
    if (!(d_k == 64 || d_k == 128) || !(d_v == 64 || d_v == 128)) return 0;
    if (!(chunk == 64 || chunk == 128)) return 0;
    if (in_dtype != ESC_DTYPE_BF16) return 0;
    if (!(out_dtype == ESC_DTYPE_F32 || out_dtype == ESC_DTYPE_BF16)) return 0;
    return (kKeyTag << 56) | ((uint64_t)B << 40) | ((uint64_t)H << 28) | ((uint64_t)(d_k / 8) << 20) |
           ((uint64_t)(d_v / 8) << 12) | ((uint64_t)in_dtype << 10) | ((uint64_t)out_dtype << 8) | (uint64_t)(chunk / 8);
}

int esc_linattn_scan(esc_ctx* ctx, esc_shape_key key, const void* q, const void* k, const void* v, const float* g,
                     const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride, uint32_t chunk,
                     void* stream) {
    ScanShape s;
    if (!ctx || !decode_key(key, &s)) return ESC_ERR_INVALID;
    if (!state_out) return ESC_ERR_INVALID;
    if (T > 0 && (!q || !k || !v || !g || !o)) return ESC_ERR_INVALID;
    if (chunk != s.chunk) return ESC_ERR_MISMATCH;
    if (t_stride < T) return ESC_ERR_INVALID;
    const uintptr_t all = (uintptr_t)q | (uintptr_t)k | (uintptr_t)v | (uintptr_t)state_in | (uintptr_t)state_out |
                          (uintptr_t)o;
    if ((all & 15u) || ((uintptr_t)g & 3u)) return ESC_ERR_UNALIGNED;  // g is read element-wise: 4-B alignment
    return launch_scan(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, (cudaStream_t)stream);
}

}  // extern "C"
