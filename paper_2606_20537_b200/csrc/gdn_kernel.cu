// Short causal convolution with carried window, and the C entry points of the gated delta-rule row (include/esc.h:
// esc_gdn_scan, esc_causal_conv) — SURVEY.md §8(f) #1: the recurrence and the convolution state of the paper's actual
// hybrid-model family ("recurrent state and convolution state are a fold over the entire prefix [4, 13]";
// DESIGN.md reading 25).  The delta-rule kernel itself is gdn_scan_kernel.cu.
#include <cuda_bf16.h>
#include <string.h>

#include "esc_internal.h"
#include "sm100_ptx.cuh"

namespace esc {

__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- short causal depthwise convolution, window W <= 8 -----------------------------------------------------
// Bound: HBM (2 B read + 4 B written per element).  A thread owns 4 consecutive channels (one 8-byte bf16 vector; a
// warp reads 256 contiguous bytes of a token row) and walks kConvRun consecutive tokens with the W-1 previous input
// vectors and its 4 x W taps in registers, so every input vector is loaded once per run (+ W-1 to prime the window).
// The loads go through a per-thread ring in shared memory filled by cp.async (kConvRing batches of kConvU vectors; a thread
// copies and reads only its OWN slots, so there is no barrier, only cp.async.wait_group): kConvRing - 1 batches are in flight
// per thread without being held in registers.  History at 16 448 x 6144, W = 4: issue -> wait -> compute -> store 150 us; the
// next batch loaded into registers before the current one is computed 113 us (r01u); packed fp32 and the fused window write
// 106.5-108.5 us; the ring 104.4 us (three, four and six batches the same, eight slower: shared memory then limits the CTAs per
// SM); runs of 48 tokens instead of 64 (four waves of shorter CTAs: the SMs idled 7 % of the launch at its ramp and tail)
// 102.4 us = 5.92 TB/s.
// SiLU is s / (1 + e^-s) with ex2.approx and the approximate divide (2 ulp each; the full-precision expf + IEEE divide
// made the kernel ALU-bound: 150 -> 120 us on their own); for s < -88 the quotient is -0 where the exact value is ~ -1e-37.
constexpr int kConvMaxW = 8;
constexpr int kConvRun = 48;      // tokens per thread (long calls; short calls take shorter runs, see conv_run_tokens)
constexpr int kConvThreads = 128;
constexpr int kConvCPT = 4;       // channels per thread (8-byte bf16 vectors: a warp reads 256 contiguous bytes of a token row)
constexpr int kConvU = 4;         // vectors per batch (one batch in flight per thread while the previous one is computed)
constexpr int kConvRing = 4;      // batches in a thread's shared-memory ring (kConvRing - 1 in flight)

__device__ __forceinline__ void bf16x4_to_f32(const uint2& raw, float (&x)[4]) {
    x[0] = __uint_as_float(raw.x << 16); x[1] = __uint_as_float(raw.x & 0xFFFF0000u);
    x[2] = __uint_as_float(raw.y << 16); x[3] = __uint_as_float(raw.y & 0xFFFF0000u);
}
__device__ __forceinline__ uint2 ld_stream8(const __nv_bfloat16* p) {
    uint2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "l"(p));
    return r;
}

template <int W>
__global__ void __launch_bounds__(kConvThreads) esc_causal_conv_kernel(const __nv_bfloat16* __restrict__ x, const float* __restrict__ w,
                                                                       const float* __restrict__ state_in, float* __restrict__ y,
                                                                       uint64_t T, uint64_t t_stride, uint32_t C, uint32_t silu, uint32_t run,
                                                                       float* state_out) {
    constexpr int P = kConvCPT, U = kConvU;
    // programmatic dependent launch: the next kernel of the stream may be placed while this one runs; this kernel touches global
    // memory only after its predecessor has completed
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const uint32_t cg = blockIdx.x * kConvThreads + threadIdx.x;   // channel group
    if (cg >= C / P) return;
    const uint32_t b = blockIdx.z;
    const uint64_t t_begin = (uint64_t)blockIdx.y * run;
    const uint32_t n_tok = (uint32_t)(t_begin + run < T ? run : T - t_begin);
    const __nv_bfloat16* xp = x + ((size_t)b * t_stride + t_begin) * C + cg * P;
    float* yp = y + ((size_t)b * T + t_begin) * C + cg * P;
    // a ring of NBR batches per thread in shared memory, filled by cp.async: each thread copies and reads its OWN slots (no
    // barrier, only cp.async.wait_group), NBR - 1 batches in flight without holding them in registers
    constexpr int NBR = kConvRing;
    __shared__ uint2 ring[NBR * U * kConvThreads];
    uint2* my = ring + threadIdx.x;
    auto issue = [&](uint32_t batch) {   // tokens [U batch, U batch + U) of the run into slot batch % NBR
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (batch * U + u < n_tok) ptx::cp_async_8(my + ((batch % NBR) * U + u) * kConvThreads, xp + (size_t)(batch * U + u) * C);
        ptx::cp_async_commit();
    };
#pragma unroll
    for (int bb = 0; bb < NBR - 1; ++bb) issue(bb);
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
            bf16x4_to_f32(ld_stream8(x + ((size_t)b * t_stride + (uint64_t)s) * C + cg * P), win[i]);
        } else {
#pragma unroll
            for (int j = 0; j < P; ++j)
                win[i][j] = state_in ? state_in[((size_t)b * C + cg * P + j) * (W - 1) + (uint32_t)((int64_t)(W - 1) + s)] : 0.f;
        }
    }
    for (uint32_t t = 0; t < n_tok; t += U) {
        uint2 raw[U];
        const uint32_t bi = t / U;
        issue(bi + NBR - 1);                  // into the slot batch bi - 1 was read from (its values are consumed)
        ptx::cp_async_wait_group<NBR - 1>();  // batch bi has landed
#pragma unroll
        for (int u = 0; u < U; ++u) raw[u] = my[((bi % NBR) * U + u) * kConvThreads];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (t + u < n_tok) {
                bf16x4_to_f32(raw[u], win[W - 1]);
                // two channels per instruction (sm_100 packed fp32: FFMA2 / FMUL2 / FADD2); same roundings as the scalar forms
                float acc[P];
#pragma unroll
                for (int j = 0; j < P; j += 2) {
                    float2 s2 = make_float2(0.f, 0.f);
#pragma unroll
                    for (int i = 0; i < W; ++i) s2 = ffma2(make_float2(wt[i][j], wt[i][j + 1]), make_float2(win[i][j], win[i][j + 1]), s2);
                    if (silu) {   // s / (1 + e^-s), e^-s = 2^(-s log2 e)
                        const float2 t = fmul2(s2, make_float2(-1.4426950408889634f, -1.4426950408889634f));
                        const float2 d = fadd2(make_float2(ex2(t.x), ex2(t.y)), make_float2(1.f, 1.f));
                        s2 = fmul2(s2, make_float2(rcp_approx(d.x), rcp_approx(d.y)));
                    }
                    acc[j] = s2.x;
                    acc[j + 1] = s2.y;
                }
                *reinterpret_cast<float4*>(yp + (size_t)u * C) = make_float4(acc[0], acc[1], acc[2], acc[3]);
#pragma unroll
                for (int i = 0; i < W - 1; ++i)
#pragma unroll
                    for (int j = 0; j < P; ++j) win[i][j] = win[i + 1][j];
            }
        }
        yp += (size_t)U * C;
    }
    // The carried window after the call (the last W-1 inputs, T >= W-1: the host passes state_out only then), written by the threads
    // of the FIRST run: they are the only ones that read state_in (a run is at least W-1 tokens long), and they have read it by
    // now, so state_out may alias state_in.  (One launch instead of two for the 64-token suffix call.)
    // (Loading these W-1 vectors up front, with the thread's other loads, saves a memory round trip on a 64-token call — 5.3 -> 5.1 us
    // chained — but costs 8 registers and a CTA of occupancy on long calls.)
    if (state_out != nullptr && blockIdx.y == 0) {
#pragma unroll
        for (int i = 0; i < W - 1; ++i) {
            float v4[P];
            bf16x4_to_f32(ld_stream8(x + ((size_t)b * t_stride + (T - (uint64_t)(W - 1) + i)) * C + cg * P), v4);
#pragma unroll
            for (int j = 0; j < P; ++j) state_out[((size_t)b * C + cg * P + j) * (W - 1) + i] = v4[j];
        }
    }
}

typedef void (*ConvKernelFn)(const __nv_bfloat16*, const float*, const float*, float*, uint64_t, uint64_t, uint32_t, uint32_t, uint32_t, float*);

// Tokens a thread walks.  64 for long calls (every input vector loaded once, + W-1 to prime the window).  A short call (the suffix
// after a restore: 64 tokens) would then be 12 CTAs walking 64 tokens one after the other: 21 us, all of it latency.  Short calls
// take runs of as few as 4 tokens (one batch in flight), so that the grid still has a few CTAs per SM: the extra priming loads hit L2.
// The arithmetic of an output does not depend on the run it falls in: same bits.
static uint32_t conv_run_tokens(uint32_t B, uint64_t T, uint32_t C, uint32_t W, uint32_t sm_count) {
    const uint64_t col_blocks = (C / kConvCPT + kConvThreads - 1) / kConvThreads;
    const uint64_t want = 4ull * (sm_count ? sm_count : 148u);                  // CTAs
    uint64_t run = (T * col_blocks * B) / want;                                  // tokens per run that give `want` CTAs
    run = run / kConvU * kConvU;
    const uint64_t run_min = (W - 1 + kConvU - 1) / kConvU * kConvU;   // >= W-1: only the first run reaches back into the carried window
    if (run < run_min) run = run_min;
    if (run < (uint64_t)kConvU) run = kConvU;
    if (run > (uint64_t)kConvRun) run = kConvRun;
    return (uint32_t)run;
}
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
    ESC_ON_DEVICE(ctx);
    return launch_gdn_mma(ctx, s, q, k, v, g, beta, state_in, state_out, (float*)o, T, t_stride, (cudaStream_t)stream);
}

int esc_causal_conv(esc_ctx* ctx, const void* x, const float* w, const float* state_in, float* state_out, float* y, uint32_t B,
                    uint64_t T, uint64_t t_stride, uint32_t C, uint32_t W, uint32_t flags, void* stream) {
    if (!ctx || !w || !state_out || B == 0 || C == 0 || t_stride < T || (flags & ~ESC_CONV_SILU)) return ESC_ERR_INVALID;
    if (T > 0 && (!x || !y)) return ESC_ERR_INVALID;
    if (W < 1 || W > (uint32_t)kConvMaxW || (C % 8) != 0) return ESC_ERR_UNSUPPORTED;
    if ((((uintptr_t)x | (uintptr_t)y) & 15u) || (((uintptr_t)w | (uintptr_t)state_in | (uintptr_t)state_out) & 3u)) return ESC_ERR_UNALIGNED;
    if (T > 0 && B > 65535) return ESC_ERR_UNSUPPORTED;
    ESC_ON_DEVICE(ctx);
    const bool fused_state = W > 1 && T >= W - 1;   // the conv kernel's first run writes the carried window itself
    if (T > 0) {
        const uint32_t run = conv_run_tokens(B, T, C, W, (uint32_t)ctx->sm_count);
        dim3 grid((C / kConvCPT + kConvThreads - 1) / kConvThreads, (uint32_t)((T + run - 1) / run), B);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grid;
        cfg.blockDim = dim3(kConvThreads);
        cfg.stream = (cudaStream_t)stream;
        cudaLaunchAttribute attr[1];
        memset(attr, 0, sizeof attr);
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddepcontrol.* in the kernel
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        ESC_CUDA(cudaLaunchKernelEx(&cfg, conv_kernel_for(W), (const __nv_bfloat16*)x, w, state_in, y, T, t_stride, C,
                                    (uint32_t)(flags & ESC_CONV_SILU), run, fused_state ? state_out : (float*)nullptr));
    }
    if (W > 1 && !fused_state && (T > 0 || state_in != state_out)) {
        const uint64_t n = (uint64_t)B * C;
        esc_conv_state_kernel<<<(uint32_t)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>((const __nv_bfloat16*)x, state_in, state_out, B, T,
                                                                                           t_stride, C, W);
        ESC_CUDA(cudaGetLastError());
    }
    return ESC_OK;
}

}  // extern "C"
