// Gated delta-rule scan and short causal convolution with carried window (include/esc.h: esc_gdn_scan,
// esc_causal_conv) — SURVEY.md §8(f) #1: the recurrence and the convolution state of the paper's actual hybrid-model
// family ("recurrent state and convolution state are a fold over the entire prefix [4, 13]"; DESIGN.md
// reading 25).
//
//     u_t = k_t (a_t S_{t-1}) ,  S_t = a_t S_{t-1} + beta_t k_t^T (v_t - u_t) ,  o_t = q_t S_t
//
// v0 of this row: the plain token-sequential form in fp32 on the CUDA cores — correct first, one code path for every T,
// so restore + continue is bit-identical to the cold run at ANY boundary (no chunk grid).  The columns of S are
// independent: one WARP owns (b, h, 4 columns of d_v) with lane l holding rows [l d_k/32, (l+1) d_k/32) of that
// [d_k x 4] slice in registers; the four warps of a CTA (16 columns) share the staged inputs and never synchronise
// inside a 64-token block.  Per token a warp needs two d_k-long dot products per column (u_t before the update, o_t after
// it); o_t and u_{t+1} both read S_t, so they share ONE warp reduction per token (8 values: transposed butterfly, 9 shuffles
// in 5 dependent steps, fixed order -> deterministic), followed by 4 broadcast shuffles.  q, k, v, a, beta are staged 64
// tokens at a time with cp.async, double buffered.  Bound: the per-token dependency chain (~250 cycles), not HBM; the
// chunked tensor-core form (WY representation + an intra-chunk triangular solve) is the next step for this row.
#include <cuda_bf16.h>

#include "esc_internal.h"

namespace esc {

constexpr int kGdnDVT = 16;       // d_v columns per CTA
constexpr int kGdnWC = 4;         // d_v columns per warp
constexpr int kGdnTB = 64;        // tokens per staged block
constexpr int kGdnThreads = 32 * (kGdnDVT / kGdnWC);

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int DK>
struct GdnSmem {
    __nv_bfloat16 q[2][kGdnTB][DK];
    __nv_bfloat16 k[2][kGdnTB][DK];
    __nv_bfloat16 v[2][kGdnTB][kGdnDVT];
    float a[2][kGdnTB];
    float beta[2][kGdnTB];
};

// Sum over the 32 lanes of 8 values per lane.  Returns the total of value index 4*bit4 + 2*bit3 + bit2 of the lane id
// (lanes 0-3 hold value 0, lanes 4-7 value 1, lanes 8-11 value 2, ..., lanes 28-31 value 7).
__device__ __forceinline__ float warp_reduce8(float (&x)[8], int lane) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float send = (lane & 16) ? x[i] : x[i + 4];
        const float keep = (lane & 16) ? x[i + 4] : x[i];
        x[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const float send = (lane & 8) ? x[i] : x[i + 2];
        const float keep = (lane & 8) ? x[i + 2] : x[i];
        x[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
    {
        const float send = (lane & 4) ? x[0] : x[1];
        const float keep = (lane & 4) ? x[1] : x[0];
        x[0] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
    x[0] += __shfl_xor_sync(0xffffffffu, x[0], 2);
    x[0] += __shfl_xor_sync(0xffffffffu, x[0], 1);
    return x[0];
}

template <int DK>
__global__ void __launch_bounds__(kGdnThreads) esc_gdn_scan_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ k,
                                                                   const __nv_bfloat16* __restrict__ v, const float* __restrict__ g,
                                                                   const float* __restrict__ beta, const float* state_in, float* state_out,
                                                                   float* __restrict__ o, uint32_t H, uint32_t DV, uint64_t T,
                                                                   uint64_t t_stride) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    GdnSmem<DK>& sm = *reinterpret_cast<GdnSmem<DK>*>(smem_raw);
    static_assert(DK == 64 || DK == 128, "d_k");
    constexpr int RPL = DK / 32;           // state rows per lane
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t bh = blockIdx.y, b = bh / H, h = bh % H, dv0 = blockIdx.x * kGdnDVT, wc0 = warp * kGdnWC;
    const int row0 = lane * RPL;

    float S[RPL][kGdnWC];
#pragma unroll
    for (int i = 0; i < RPL; ++i) {
        float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
        if (state_in) x = *reinterpret_cast<const float4*>(state_in + ((size_t)bh * DK + row0 + i) * DV + dv0 + wc0);
        S[i][0] = x.x; S[i][1] = x.y; S[i][2] = x.z; S[i][3] = x.w;
    }

    const uint64_t n_blocks = (T + kGdnTB - 1) / kGdnTB;
    auto stage = [&](uint64_t blk, int buf) {   // tokens [blk*TB, ...) -> buffer buf (rows beyond T are not loaded nor used)
        const uint64_t t0 = blk * kGdnTB;
        const int n = (int)((T - t0) < (uint64_t)kGdnTB ? (T - t0) : (uint64_t)kGdnTB);
        constexpr int CH = DK / 8;                      // 16-byte pieces per token row of q / k
        for (int i = tid; i < n * CH; i += kGdnThreads) {
            const int tt = i / CH, c = i % CH;
            const size_t tok = ((size_t)b * t_stride + t0 + tt) * H + h;
            cp_async16(&sm.q[buf][tt][c * 8], q + tok * DK + c * 8);
            cp_async16(&sm.k[buf][tt][c * 8], k + tok * DK + c * 8);
        }
        for (int i = tid; i < n * 2; i += kGdnThreads) {
            const size_t tok = ((size_t)b * t_stride + t0 + (i >> 1)) * H + h;
            cp_async16(&sm.v[buf][i >> 1][(i & 1) * 8], v + tok * DV + dv0 + (i & 1) * 8);
        }
        for (int i = tid; i < n; i += kGdnThreads) {
            const size_t tok = ((size_t)b * t_stride + t0 + i) * H + h;
            cp_async4(&sm.a[buf][i], g + tok);
            cp_async4(&sm.beta[buf][i], beta + tok);
        }
        cp_async_commit();
    };
    auto load_rows = [&](const __nv_bfloat16* p, float (&x)[RPL]) {   // RPL consecutive bf16 of a staged row -> fp32
        if constexpr (RPL == 4) {
            const uint2 w = *reinterpret_cast<const uint2*>(p + row0);
            x[0] = __uint_as_float(w.x << 16); x[1] = __uint_as_float(w.x & 0xFFFF0000u);
            x[2] = __uint_as_float(w.y << 16); x[3] = __uint_as_float(w.y & 0xFFFF0000u);
        } else {
            const uint32_t w = *reinterpret_cast<const uint32_t*>(p + row0);
            x[0] = __uint_as_float(w << 16); x[1] = __uint_as_float(w & 0xFFFF0000u);
        }
    };

    if (n_blocks) stage(0, 0);
    for (uint64_t blk = 0; blk < n_blocks; ++blk) {
        const int buf = (int)(blk & 1);
        if (blk + 1 < n_blocks) {
            stage(blk + 1, buf ^ 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
        const uint64_t t0 = blk * kGdnTB;
        const int n = (int)((T - t0) < (uint64_t)kGdnTB ? (T - t0) : (uint64_t)kGdnTB);
        float part[8], kr[RPL], qr[RPL], kn[RPL];
        // r_t = k_t . S_{t-1} for the first token of the block (every later r comes out of the previous token's reduction)
        load_rows(&sm.k[buf][0][0], kr);
#pragma unroll
        for (int j = 0; j < kGdnWC; ++j) {
            float acc = 0.f;
#pragma unroll
            for (int i = 0; i < RPL; ++i) acc = fmaf(kr[i], S[i][j], acc);
            part[j] = acc;
            part[4 + j] = 0.f;
        }
        float tot = warp_reduce8(part, lane);
        float r[kGdnWC];
#pragma unroll
        for (int j = 0; j < kGdnWC; ++j) r[j] = __shfl_sync(0xffffffffu, tot, 4 * j);   // value j lives in lanes 4j .. 4j+3
        for (int tt = 0; tt < n; ++tt) {
            load_rows(&sm.q[buf][tt][0], qr);
            const bool more = tt + 1 < n;
            if (more) load_rows(&sm.k[buf][tt + 1][0], kn);
            const float a = sm.a[buf][tt], bt = sm.beta[buf][tt];
            const uint2 vraw = *reinterpret_cast<const uint2*>(&sm.v[buf][tt][wc0]);
            const float vj[4] = {__uint_as_float(vraw.x << 16), __uint_as_float(vraw.x & 0xFFFF0000u), __uint_as_float(vraw.y << 16),
                                 __uint_as_float(vraw.y & 0xFFFF0000u)};
            // S_t = a_t S_{t-1} + beta_t k_t^T (v_t - u_t), u_t = a_t r_t;  then k_{t+1} . S_t and q_t . S_t in ONE reduction
#pragma unroll
            for (int j = 0; j < kGdnWC; ++j) {
                const float wj = bt * (vj[j] - a * r[j]);
                float pk = 0.f, pq = 0.f;
#pragma unroll
                for (int i = 0; i < RPL; ++i) {
                    S[i][j] = fmaf(kr[i], wj, a * S[i][j]);
                    pk = fmaf(more ? kn[i] : 0.f, S[i][j], pk);
                    pq = fmaf(qr[i], S[i][j], pq);
                }
                part[j] = pk;
                part[4 + j] = pq;
            }
            tot = warp_reduce8(part, lane);
#pragma unroll
            for (int j = 0; j < kGdnWC; ++j) r[j] = __shfl_sync(0xffffffffu, tot, 4 * j);
            if (lane >= 16 && (lane & 3) == 0)   // lanes 16, 20, 24, 28 hold o_t of columns 0..3 of this warp
                o[(((size_t)b * t_stride + t0 + tt) * H + h) * DV + dv0 + wc0 + ((lane - 16) >> 2)] = tot;
#pragma unroll
            for (int i = 0; i < RPL; ++i) kr[i] = kn[i];
        }
        __syncthreads();   // everyone is done with buffer `buf` before it is staged again
    }
#pragma unroll
    for (int i = 0; i < RPL; ++i)
        *reinterpret_cast<float4*>(state_out + ((size_t)bh * DK + row0 + i) * DV + dv0 + wc0) = make_float4(S[i][0], S[i][1], S[i][2], S[i][3]);
}

// ---- short causal depthwise convolution, window W <= 8 -----------------------------------------------------
// Bound: HBM (2 B read + 4 B written per element).  A thread owns 4 consecutive channels (one 8-byte bf16 vector; a
// warp reads 256 contiguous bytes of a token row) and walks kConvRun consecutive tokens with the W-1 previous input
// vectors and its 8 x W taps in registers, so every input vector is loaded once per run (+ W-1 to prime the window).
constexpr int kConvMaxW = 8;
constexpr int kConvRun = 64;      // tokens per thread
constexpr int kConvThreads = 128;
constexpr int kConvCPT = 4;       // channels per thread (8-byte bf16 vectors: a warp reads 256 contiguous bytes of a token row)

__device__ __forceinline__ void bf16x4_to_f32(const uint2& raw, float (&x)[4]) {
    x[0] = __uint_as_float(raw.x << 16); x[1] = __uint_as_float(raw.x & 0xFFFF0000u);
    x[2] = __uint_as_float(raw.y << 16); x[3] = __uint_as_float(raw.y & 0xFFFF0000u);
}

template <int W>
__global__ void __launch_bounds__(kConvThreads) esc_causal_conv_kernel(const __nv_bfloat16* __restrict__ x, const float* __restrict__ w,
                                                                       const float* __restrict__ state_in, float* __restrict__ y,
                                                                       uint64_t T, uint64_t t_stride, uint32_t C, uint32_t silu) {
    constexpr int P = kConvCPT;
    const uint32_t cg = blockIdx.x * kConvThreads + threadIdx.x;   // channel group
    if (cg >= C / P) return;
    const uint32_t b = blockIdx.z;
    const uint64_t t_begin = (uint64_t)blockIdx.y * kConvRun;
    const uint64_t t_end = t_begin + kConvRun < T ? t_begin + kConvRun : T;
    float wt[W][P];   // wt[i][j] = tap i of channel P cg + j
#pragma unroll
    for (int j = 0; j < P; ++j)
#pragma unroll
        for (int i = 0; i < W; ++i) wt[i][j] = w[(size_t)(cg * P + j) * W + i];
    // win[i] = input at position t - (W-1) + i for the current t; primed with the W-1 inputs before t_begin
    float win[W][P];
#pragma unroll
    for (int i = 0; i < W - 1; ++i) {
        const int64_t s = (int64_t)t_begin - (W - 1) + i;
        if (s >= 0) {
            bf16x4_to_f32(*reinterpret_cast<const uint2*>(x + ((size_t)b * t_stride + (uint64_t)s) * C + cg * P), win[i]);
        } else {
#pragma unroll
            for (int j = 0; j < P; ++j)
                win[i][j] = state_in ? state_in[((size_t)b * C + cg * P + j) * (W - 1) + (uint32_t)((int64_t)(W - 1) + s)] : 0.f;
        }
    }
    const __nv_bfloat16* xp = x + ((size_t)b * t_stride + t_begin) * C + cg * P;
    float* yp = y + ((size_t)b * T + t_begin) * C + cg * P;
    constexpr int U = 4;   // loads in flight per thread
    for (uint64_t t = t_begin; t < t_end; t += U) {
        uint2 raw[U];
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (t + u < t_end) raw[u] = *reinterpret_cast<const uint2*>(xp + (size_t)u * C);
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (t + u < t_end) {
                bf16x4_to_f32(raw[u], win[W - 1]);
                float acc[P];
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    float s_ = 0.f;
#pragma unroll
                    for (int i = 0; i < W; ++i) s_ = fmaf(wt[i][j], win[i][j], s_);
                    acc[j] = silu ? s_ / (1.f + expf(-s_)) : s_;
                }
                *reinterpret_cast<float4*>(yp + (size_t)u * C) = make_float4(acc[0], acc[1], acc[2], acc[3]);
#pragma unroll
                for (int i = 0; i < W - 1; ++i)
#pragma unroll
                    for (int j = 0; j < P; ++j) win[i][j] = win[i + 1][j];
            }
        }
        xp += (size_t)U * C;
        yp += (size_t)U * C;
    }
}

typedef void (*ConvKernelFn)(const __nv_bfloat16*, const float*, const float*, float*, uint64_t, uint64_t, uint32_t, uint32_t);
static ConvKernelFn conv_kernel_for(uint32_t W) {
    switch (W) {
        case 1: return esc_causal_conv_kernel<1>;
        case 2: return esc_causal_conv_kernel<2>;
        case 3: return esc_causal_conv_kernel<3>;
        case 4: return esc_causal_conv_kernel<4>;
        case 5: return esc_causal_conv_kernel<5>;
        case 6: return esc_causal_conv_kernel<6>;
        case 7: return esc_causal_conv_kernel<7>;
        case 8: return esc_causal_conv_kernel<8>;
    }
    return nullptr;
}

// carried window after the call: the last W-1 inputs per (b, c), oldest first; one thread per (b, c), reads before it writes
__global__ void esc_conv_state_kernel(const __nv_bfloat16* __restrict__ x, const float* state_in, float* state_out, uint32_t B, uint64_t T,
                                      uint64_t t_stride, uint32_t C, uint32_t W) {
    const uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (uint64_t)B * C) return;
    const uint32_t c = (uint32_t)(idx % C), b = (uint32_t)(idx / C);
    float nv[kConvMaxW];
    for (uint32_t i = 0; i + 1 < W; ++i) {
        const int64_t s = (int64_t)T - (int64_t)(W - 1) + (int64_t)i;
        if (s >= 0) nv[i] = __bfloat162float(x[((size_t)b * t_stride + (uint64_t)s) * C + c]);
        else nv[i] = state_in ? state_in[((size_t)b * C + c) * (W - 1) + (uint32_t)((int64_t)W - 1 + s)] : 0.f;
    }
    for (uint32_t i = 0; i + 1 < W; ++i) state_out[((size_t)b * C + c) * (W - 1) + i] = nv[i];
}

template <int DK>
static int launch_gdn_t(const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* beta,
                        const float* state_in, float* state_out, float* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    static bool attr_set = false;
    if (!attr_set) {
        ESC_CUDA(cudaFuncSetAttribute(esc_gdn_scan_kernel<DK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GdnSmem<DK>)));
        attr_set = true;
    }
    dim3 grid(s.dv / kGdnDVT, s.B * s.H);
    esc_gdn_scan_kernel<DK><<<grid, kGdnThreads, sizeof(GdnSmem<DK>), stream>>>(
        (const __nv_bfloat16*)q, (const __nv_bfloat16*)k, (const __nv_bfloat16*)v, g, beta, state_in, state_out, o, s.H, s.dv, T, t_stride);
    ESC_CUDA(cudaGetLastError());
    return ESC_OK;
}

}  // namespace esc

using namespace esc;

extern "C" {

int esc_gdn_scan(esc_ctx* ctx, esc_shape_key key, const void* q, const void* k, const void* v, const float* g, const float* beta,
                 const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride, void* stream) {
    ScanShape s;
    if (!ctx || !decode_key(key, &s) || !state_out) return ESC_ERR_INVALID;
    if (T > 0 && (!q || !k || !v || !g || !beta || !o)) return ESC_ERR_INVALID;
    if (t_stride < T) return ESC_ERR_INVALID;
    if (s.out_dtype != ESC_DTYPE_F32) return ESC_ERR_UNSUPPORTED;
    const uintptr_t all = (uintptr_t)q | (uintptr_t)k | (uintptr_t)v | (uintptr_t)state_in | (uintptr_t)state_out | (uintptr_t)o;
    if ((all & 15u) || (((uintptr_t)g | (uintptr_t)beta) & 3u)) return ESC_ERR_UNALIGNED;
    if (s.dk == 128) return launch_gdn_t<128>(s, q, k, v, g, beta, state_in, state_out, (float*)o, T, t_stride, (cudaStream_t)stream);
    if (s.dk == 64) return launch_gdn_t<64>(s, q, k, v, g, beta, state_in, state_out, (float*)o, T, t_stride, (cudaStream_t)stream);
    return ESC_ERR_UNSUPPORTED;
}

int esc_causal_conv(esc_ctx* ctx, const void* x, const float* w, const float* state_in, float* state_out, float* y, uint32_t B,
                    uint64_t T, uint64_t t_stride, uint32_t C, uint32_t W, uint32_t flags, void* stream) {
    if (!ctx || !w || !state_out || B == 0 || C == 0 || t_stride < T || (flags & ~ESC_CONV_SILU)) return ESC_ERR_INVALID;
    if (T > 0 && (!x || !y)) return ESC_ERR_INVALID;
    if (W < 1 || W > (uint32_t)kConvMaxW || (C % 8) != 0) return ESC_ERR_UNSUPPORTED;
    if ((((uintptr_t)x | (uintptr_t)y) & 15u) || (((uintptr_t)w | (uintptr_t)state_in | (uintptr_t)state_out) & 3u)) return ESC_ERR_UNALIGNED;
    if (T > 0) {
        if (B > 65535) return ESC_ERR_UNSUPPORTED;
        dim3 grid((C / kConvCPT + kConvThreads - 1) / kConvThreads, (uint32_t)((T + kConvRun - 1) / kConvRun), B);
        conv_kernel_for(W)<<<grid, kConvThreads, 0, (cudaStream_t)stream>>>((const __nv_bfloat16*)x, w, state_in, y, T, t_stride, C,
                                                                            flags & ESC_CONV_SILU);
        ESC_CUDA(cudaGetLastError());
    }
    if (W > 1 && (T > 0 || state_in != state_out)) {
        const uint64_t n = (uint64_t)B * C;
        esc_conv_state_kernel<<<(uint32_t)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>((const __nv_bfloat16*)x, state_in, state_out, B, T,
                                                                                           t_stride, C, W);
        ESC_CUDA(cudaGetLastError());
    }
    return ESC_OK;
}

}  // extern "C"
