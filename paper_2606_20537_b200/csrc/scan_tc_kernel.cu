// Chunked gated linear-attention scan, sm_100a tensor-core path (include/esc.h: esc_linattn_scan).
//
// Definition (BASELINE.json north_star; "a fold over the entire prefix", folded "per
// chunk" PAPER.md:169):   S_t = g_t S_{t-1} + k_t^T v_t ,  o_t = q_t S_t.
// Chunk algebra (exact-arithmetic equivalent; every exponent <= 0), with b_i = sum_{r<=i} log2 g_r:
//     P      = Q K^T                                  (C x C)     tcgen05.mma  M=C   N=C/CS  K=d_k  (a column slice per CTA)
//     A_ij   = P_ij 2^(b_i - b_j) [j <= i]            fp32 ALU + MUFU, split into bf16 hi + lo
//     O1     = Q [S_hi | S_lo]                        (C x 32)    tcgen05.mma  M=C   N=32  K=d_k
//     O2     = A_hi V + A_lo V                        (C x 16)    tcgen05.mma  M=C   N=16  K=C  (x2)
//     o_i    = 2^(b_i) (O1h_i + O1l_i) + O2_i         fp32 epilogue
//     U      = K^T [V~_hi | V~_lo] , V~_j = 2^(b_C - b_j) v_j   (d_k x 32)  tcgen05.mma  M=d_k N=32 K=C
//     S_next = 2^(b_C) S_prev + (Uh + Ul)             fp32 FMA in registers (the carry chain)
//
// Decomposition.  The columns of S are independent, so one CTA owns (b, h, 16 columns of d_v) and walks
// the chunks in order with its state slice in registers.  CS = 4 neighbouring d_v slices of a head form a
// THREAD-BLOCK CLUSTER and share everything that does not depend on the d_v slice:
//   * Q and K tiles: CTA r loads rows [r C/CS, (r+1) C/CS) of each tile and TMA-multicasts them into the
//     same stage of all CS CTAs (L2 -> SM traffic for Q, K drops CS-fold);
//   * the scores: CTA r computes only the column slice P[:, r C/CS ...] (an N = C/CS MMA), turns it into
//     the A slice (decay, causal mask, hi/lo split) in its own A operand buffer and pushes that contiguous
//     slice into the same place of every peer's buffer with one bulk shared::cta -> shared::cluster copy
//     per peer, completing (tx bytes) on the peer's mbarrier.
// Ring and A-buffer reuse are therefore cluster-wide events: stage / A-buffer "empty" barriers count
// tcgen05.commit arrivals multicast from all CS CTAs.  The score path (P -> A -> O2) has its own buffers
// (NB of each, O2 reads V from a copy the V~ warps make), so it never holds an input stage.
// Calls of up to kTcShortT tokens use the CS = 1 instantiation instead: no cluster, every CTA loads whole Q / K tiles and
// computes all C columns of P and A itself (bit-identical results; see kTcShortT below for why).
// What bounds it (r01: ncu, clock64 traces, per-warp busy/wait accounting, ablation builds): the four MMA-issuing
// threads.  They are the busiest threads of the CTA (1200-1400 of a 1400-cycle period per chunk; every other role
// 600-1000): 28 small tcgen05.mma (M = 64, N = 16..32) and 11 tcgen05.commit per chunk at ~110 / ~130 cycles of issuing-
// thread time each, where the tensor pipe itself needs 13-23 cycles per such MMA (microbenchmark).  DRAM, tensor pipe,
// issue slots, L2, DSMEM and the TMA loads each have slack (removing any one of them changes nothing).  The d_v split
// that fills the SMs at B H = 16 is what makes the MMAs this small; DESIGN.md 6.2 lists what was tried.
//
// Warp roles (22 warps, mbarrier-synchronised software pipeline, no CTA-wide barrier in the loop):
//   warp 0         TMA producer (multicast Q/K row slices, own V slice; L2 prefetch ahead)
//   warp 1         gate warp: log2 g, segmented warp-shuffle prefix sums, 256 tokens per batch
//   warps 2,3,4,5  MMA issuers, one thread each: P | O1 | U | O2 (a tcgen05.mma costs its issuing thread
//                  ~55 cycles whatever its shape: four issuers keep the pipe, not the issue slot, the limit)
//   warps 6,7,20,21  V~ warps: V -> V~ hi/lo operand (own barrier: U and the carry never wait for scores)
//   warps 8-11     score warps (one per TMEM lane quadrant): P slice (TMEM) -> A slice -> all CTAs
//   warps 12-15    state warps: U (TMEM) -> carry S in fp32 registers -> [S_hi | S_lo] operand
//   warps 16-19    epilogue warps: O1, O2 (TMEM) -> o (global)
//   warps 22-25    second set of score warps: the upper half of the slice's key columns
//
// Bit-identity: the carry is a pure function of (S_prev bits, chunk inputs); there
// is no T-dependent tiling, no atomics, no split-K; every accumulator is produced by ONE issuer thread
// in a fixed order, every A element by one thread of one CTA.  Precision: raw Q, K, V
// are the bf16 inputs; A, V~, S_prev are two-term bf16 splits (hi + lo), the hi|lo halves of V~ and S
// ride in one MMA as 32 columns.
#include <cuda.h>
#include <cuda_bf16.h>

#include "esc_internal.h"
#include "sm100_ptx.cuh"

namespace esc {

using namespace ptx;
typedef __nv_bfloat16 bf16;

constexpr int kTcWarps = 22;
constexpr int kTcThreads = kTcWarps * 32;
// Both variants run a second set of four score warps (warps 22-25; first for the cluster-free short-call variant): each set takes half of the C key
// columns of every row quadrant, which halves the longest score warp's work on the one-chunk critical path
// (r01u, 18-layer suffix graph: 4.78 -> 4.55 us per layer; same elements by the same expressions: bit-identical).
#ifndef ESC_TC_SW
#define ESC_TC_SW 2
#endif
// The cluster variant runs the second set too (each set 8 of the slice's 16 key columns): 211 -> 207 us at 16 448 tokens,
// -2 % across the config-4 sweep, -6 % at T = 2048 (r01u).
#ifndef ESC_TC_SW_LONG
#define ESC_TC_SW_LONG 2
#endif
template <int CS> struct TcScore {
    static constexpr int sets = CS == 1 ? ESC_TC_SW : ESC_TC_SW_LONG;
    static constexpr int threads = (kTcWarps + 4 * (sets - 1)) * 32;
};
constexpr int kTcThreadsMax = (kTcWarps + 4) * 32;
constexpr int kTcDVT = 16;        // d_v columns per CTA
constexpr int kTcNM = 2 * kTcDVT; // columns of a merged hi|lo operand
constexpr int kGateBatch = 256;   // tokens per gate-warp batch
constexpr int kPrefetchAhead = 6; // chunks the producer prefetches into L2 ahead of its smem ring
constexpr int kVtThreads = 128;   // threads of the four V~ warps

#ifdef ESC_TC_TRACE   // bring-up only: per-chunk clock64() stamps of CTA (0,0), read back with esc_debug_trace_read
__device__ long long g_tc_trace[16 * 64];
__device__ unsigned int g_tc_launch;
#define TC_TRACE(ev, c) do { if (blockIdx.x == 0 && blockIdx.y == 0 && (c) < 64) g_tc_trace[(ev) * 64 + (c)] = clock64(); } while (0)
// launch-level stamps (globaltimer, ns) of CTA (0,0) thread 0, one column per launch
__device__ __forceinline__ long long tc_gtime() { long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define TC_TRACE_L(ev, id) do { if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) g_tc_trace[(ev) * 64 + ((id) & 63)] = tc_gtime(); } while (0)
#else
#define TC_TRACE(ev, c) do { } while (0)
#define TC_TRACE_L(ev, id) do { } while (0)
#endif

template <int DK, int C, int CS>
struct TcCfg {
    static constexpr int NS = (C == 64) ? 4 : 2;          // input stages
    static constexpr int NB = (C == 64) ? 3 : 1;          // P / A / V~ (+ V copy) buffers
    static constexpr int NSB = (C == 64) ? 2 : 1;         // S operand buffers
    static constexpr int NH = DK / 64;                    // 64-column halves of a Q / K tile
    static constexpr int CPB = kGateBatch / C;            // chunks per gate batch
    static constexpr uint32_t half_bytes = C * 128;       // one [C x 64] bf16 half tile
    static constexpr uint32_t q_bytes = NH * half_bytes;
    static constexpr uint32_t v_bytes = C * 32;           // [C x 16] bf16
    static constexpr uint32_t stage_bytes = 2 * q_bytes + v_bytes;   // multiple of 1024
    // A operand (M = C rows i, K = C keys j), K-major, no swizzle, hi and lo terms interleaved per 8-key group:
    //   (term, i, j) -> (j/8) a_lbo + term a_term + (i/8) 128 + (i%8) 16 + (j%8) 2
    // so that the 8-key groups of one CTA's column slice are contiguous (one bulk copy per 16-row group and term)
    static constexpr uint32_t a_term = (C / 8) * 128;     // one term of one 8-key group: [C x 8] bf16
    static constexpr uint32_t a_lbo = 2 * a_term;
    static constexpr uint32_t a_bytes = (C / 8) * a_lbo;  // both terms
    static constexpr uint32_t vc_off = C * kTcNM * 2;     // V~ buffer: merged V~ operand [32 x C], then a copy of the V tile
    static constexpr uint32_t vt_bytes = vc_off + v_bytes;
    static constexpr uint32_t s_bytes = DK * kTcNM * 2;   // merged S operand [32 x DK]
    // offsets from the 1024-aligned base
    static constexpr uint32_t stage_off = 0;
    static constexpr uint32_t a_off = stage_off + NS * stage_bytes;             // [NB]
    static constexpr uint32_t vt_off = a_off + NB * a_bytes;                    // [NB]
    static constexpr uint32_t s_off = vt_off + NB * vt_bytes;                   // [NSB]
    static constexpr uint32_t gate_off = s_off + NSB * s_bytes;                 // [2][b2[256], eb[256]] fp32
    static constexpr uint32_t bar_off = gate_off + 2 * 2 * kGateBatch * 4;
    static constexpr uint32_t n_bars = 2 * NS + 6 * NB + 2 * NSB + 14;
    static constexpr uint32_t total = bar_off + 64 * 8 + 16 + 1024;             // + alignment slack
    static constexpr uint32_t p_cols = (C / CS <= 32) ? 32 : 64;   // TMEM columns of one P buffer (a slice has C/CS keys)
    static constexpr uint32_t tm_p = 0;                    // [NB] x p_cols
    static constexpr uint32_t tm_u = NB * p_cols;          // [2] x 32
    static constexpr uint32_t tm_o1 = tm_u + 64;           // [2] x 32
    static constexpr uint32_t tm_o2 = tm_o1 + 64;          // [2] x 16
    static constexpr uint32_t tmem_cols = (tm_o2 + 32 <= 256) ? 256 : 512;
    static_assert(tm_o2 + 32 <= tmem_cols, "TMEM budget");
    static_assert(stage_bytes % 1024 == 0, "stages must keep 1024-byte alignment (128B swizzle)");
    static_assert(n_bars <= 64, "barrier area");
    static_assert(total <= 232448, "shared memory budget");
};

struct TcBars {   // indices into the mbarrier array
    int full, empty, p_full, p_empty, a_full, a_empty, vt_full, vt_empty, s_full, s_empty, o1_full, o2_full, o_empty, u_full,
        u_empty, g_full, g_empty;
};
template <int DK, int C, int CS>
__device__ __forceinline__ constexpr TcBars tc_bars() {
    using L = TcCfg<DK, C, CS>;
    TcBars b{};
    int i = 0;
    b.full = i; i += L::NS;
    b.empty = i; i += L::NS;
    b.p_full = i; i += L::NB;
    b.p_empty = i; i += L::NB;
    b.a_full = i; i += L::NB;
    b.a_empty = i; i += L::NB;
    b.vt_full = i; i += L::NB;
    b.vt_empty = i; i += L::NB;
    b.s_full = i; i += L::NSB;
    b.s_empty = i; i += L::NSB;
    b.o1_full = i; i += 2;
    b.o2_full = i; i += 2;
    b.o_empty = i; i += 2;
    b.u_full = i; i += 2;
    b.u_empty = i; i += 2;
    b.g_full = i; i += 2;
    b.g_empty = i; i += 2;
    return b;
}

__device__ __forceinline__ uint32_t pack_bf16(float lo_elem, float hi_elem) {   // element 0 in the low half
    __nv_bfloat162 p = __floats2bfloat162_rn(lo_elem, hi_elem);
    return *reinterpret_cast<uint32_t*>(&p);
}
// two-term split of a pair: returns packed hi terms, writes packed lo terms
__device__ __forceinline__ uint32_t split2(float x0, float x1, uint32_t& lo) {
    const uint32_t hi = pack_bf16(x0, x1);   // one cvt.rn.bf16x2.f32
    lo = pack_bf16(x0 - __uint_as_float(hi << 16), x1 - __uint_as_float(hi & 0xFFFF0000u));
    return hi;
}
__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <typename OutT>
__device__ __forceinline__ void store_o2(OutT* p, float x0, float x1);
template <>
__device__ __forceinline__ void store_o2<float>(float* p, float x0, float x1) {
    *reinterpret_cast<float2*>(p) = make_float2(x0, x1);
}
template <>
__device__ __forceinline__ void store_o2<bf16>(bf16* p, float x0, float x1) {
    *reinterpret_cast<uint32_t*>(p) = pack_bf16(x0, x1);
}

// 16 TMEM lanes x NA fp32 columns -> NA/2 registers per thread (layout: see tmem_ld_16x256b_x2 in sm100_ptx.cuh)
template <int NA>
__device__ __forceinline__ void tmem_ld_slice(uint32_t addr, uint32_t* r) {
    if constexpr (NA == 8) tmem_ld_16x256b_x1(addr, r);
    else if constexpr (NA == 16) tmem_ld_16x256b_x2(addr, r);
    else if constexpr (NA == 32) tmem_ld_16x256b_x4(addr, r);
    else tmem_ld_16x256b_x8(addr, r);
}

template <int DK, int C, int CS, typename OutT>
__global__ void __launch_bounds__(kTcThreadsMax, 1)
esc_scan_tc_kernel(const __grid_constant__ CUtensorMap tq, const __grid_constant__ CUtensorMap tk,
                   const __grid_constant__ CUtensorMap tv, const float* __restrict__ g, const float* state_in,
                   float* state_out, OutT* __restrict__ o, uint32_t H, uint32_t DV, uint64_t T, uint64_t t_stride) {
    using L = TcCfg<DK, C, CS>;
    constexpr TcBars BI = tc_bars<DK, C, CS>();
    constexpr int NS = L::NS, NB = L::NB, NSB = L::NSB, CPB = L::CPB;
    constexpr int NA = C / CS;                      // keys per score slice = Q / K rows this CTA loads
    constexpr int SW = TcScore<CS>::sets;           // score-warp sets (each takes NA / SW of the slice's key columns)
    constexpr int NAW = NA / SW;
    constexpr uint16_t kAll = (uint16_t)((1u << CS) - 1);
    constexpr uint32_t SBO_V = (C / 8) * 128, SBO_S = (DK / 8) * 128;
    static_assert(NA == 8 || NA == 16 || NA == 32 || NA == 64, "slice width");
    static_assert(C == 128 ? NA >= 16 : true, "an M = 128 MMA needs N % 16 == 0");

    extern __shared__ uint8_t smem_raw[];
    uint8_t* sm = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // same offset in every CTA of the cluster
    const uint32_t sm_a = smem_u32(sm);
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + L::bar_off);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sm + L::bar_off + 64 * 8);
    float* gate = reinterpret_cast<float*>(sm + L::gate_off);   // [2][2][256]: b2 then eb per slot

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t rank = 0;
    if constexpr (CS > 1) rank = cluster_ctarank();   // clusters are CS consecutive d_v slices (blockIdx.x) of one (b, h)
    const uint32_t bh = blockIdx.y, b = bh / H, h = bh % H, dv0 = blockIdx.x * kTcDVT;
    const uint32_t key0 = rank * NA;    // first key (= first Q / K row) of this CTA's slice
    const uint32_t n_chunks = (uint32_t)((T + C - 1) / C);
    const int q = warp & 3;   // TMEM lane quadrant this warp may access
    if (threadIdx.x == 0) TC_TRACE(9, 0);
#ifdef ESC_TC_TRACE
    unsigned int launch_id = 0;
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) launch_id = atomicAdd(&g_tc_launch, 1u);
    TC_TRACE_L(13, launch_id);
#endif
    // Programmatic dependent launch: the next kernel of the stream / graph (typically the next layer's scan) may start
    // its on-chip setup while this one runs; everything this kernel reads from or writes to global memory comes after
    // griddepcontrol.wait below, i.e. after the preceding kernel has completed and flushed.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    // commit that every CTA of the cluster must see (stage / A-buffer reuse)
    auto commit_all = [&](uint64_t* bar) {
        if constexpr (CS > 1) mma_commit_mc(bar, kAll);
        else mma_commit(bar);
    };
    // TMA producer steps (warp 0, lane 0)
    auto tma_prefetch_chunk = [&](uint32_t c) {   // pull this CTA's share of chunk c into L2
        const int t0 = (int)(c * C);
        if constexpr (CS == 1) {
            tma_prefetch_5d(&tq, 0, t0, 0, (int)h, (int)b);
            tma_prefetch_5d(&tk, 0, t0, 0, (int)h, (int)b);
        } else {
#pragma unroll
            for (int hh = 0; hh < L::NH; ++hh) {
                tma_prefetch_4d(&tq, hh * 64, (int)h, t0 + (int)key0, (int)b);
                tma_prefetch_4d(&tk, hh * 64, (int)h, t0 + (int)key0, (int)b);
            }
        }
        tma_prefetch_4d(&tv, (int)dv0, (int)h, t0, (int)b);
    };
    auto tma_issue = [&](uint32_t c) {   // chunk c -> stage c % NS of ALL CTAs (Q, K rows key0..) / of this CTA (V)
        const uint32_t s = c % NS;
        uint8_t* st = sm + L::stage_off + s * L::stage_bytes;
        uint64_t* full = &bars[BI.full + s];
        mbar_arrive_expect_tx(full, L::stage_bytes);   // Q and K arrive in CS row slices, one from each CTA
        const int t0 = (int)(c * C);
        if constexpr (CS > 1) {
#pragma unroll
            for (int hh = 0; hh < L::NH; ++hh) {
                tma_load_4d_mc(st + hh * L::half_bytes + key0 * 128, &tq, full, hh * 64, (int)h, t0 + (int)key0, (int)b, kAll);
                tma_load_4d_mc(st + L::q_bytes + hh * L::half_bytes + key0 * 128, &tk, full, hh * 64, (int)h, t0 + (int)key0, (int)b,
                               kAll);
            }
        } else {
            // on its own a CTA takes a whole tile per instruction: the map has the 64-column halves as its third dimension
            // (d % 64, t, d / 64, h, b), so a box of (64, C, NH) lands as [half][token][64] — the two half tiles back to back
            // (r01u trace: the producer needs ~200 cycles per TMA instruction, and a one-chunk call waits for all of them)
            tma_load_5d(st, &tq, full, 0, t0, 0, (int)h, (int)b);
            tma_load_5d(st + L::q_bytes, &tk, full, 0, t0, 0, (int)h, (int)b);
        }
        tma_load_4d(st + 2 * L::q_bytes, &tv, full, (int)dv0, (int)h, t0, (int)b);
        TC_TRACE(0, c);
    };

    // ---- one-time setup, on-chip part (under programmatic dependent launch it overlaps the preceding kernel) -----------
    if (warp == 0 && lane == 0) {
        for (int i = 0; i < NS; ++i) { mbar_init(&bars[BI.full + i], 1); mbar_init(&bars[BI.empty + i], 3 * CS); }
        for (int i = 0; i < NB; ++i) {
            mbar_init(&bars[BI.p_full + i], 1); mbar_init(&bars[BI.p_empty + i], 4 * SW);
            mbar_init(&bars[BI.a_full + i], 4 * SW); mbar_init(&bars[BI.a_empty + i], CS);
            mbar_init(&bars[BI.vt_full + i], 4); mbar_init(&bars[BI.vt_empty + i], 2);
        }
        for (int i = 0; i < NSB; ++i) { mbar_init(&bars[BI.s_full + i], 4); mbar_init(&bars[BI.s_empty + i], 1); }
        for (int i = 0; i < 2; ++i) {
            mbar_init(&bars[BI.o1_full + i], 1); mbar_init(&bars[BI.o2_full + i], 1); mbar_init(&bars[BI.o_empty + i], 4);
            mbar_init(&bars[BI.u_full + i], 1); mbar_init(&bars[BI.u_empty + i], 4);
            mbar_init(&bars[BI.g_full + i], 1); mbar_init(&bars[BI.g_empty + i], 16 + 4 * (SW - 1));
        }
        fence_mbar_init();
        tma_prefetch_desc(&tq); tma_prefetch_desc(&tk); tma_prefetch_desc(&tv);
    }
    if (warp == 2) tmem_alloc(tmem_slot, L::tmem_cols);
    // A buffers: blocks above the causal diagonal are never written by any CTA and must read as zero
    // (a CTA on its own, CS = 1, writes every element of A itself, the masked ones as zeros)
    if constexpr (CS > 1) {
        for (uint32_t i = threadIdx.x; i < NB * L::a_bytes / 16; i += kTcThreads)
            reinterpret_cast<uint4*>(sm + L::a_off)[i] = make_uint4(0, 0, 0, 0);
    }
    fence_proxy_async_smem();
    tc_fence_before_sync();
    // every CTA's barriers are initialised and its A buffers zeroed before any peer multicasts / copies into them
    if constexpr (CS > 1) cluster_sync();
    else __syncthreads();
    tc_fence_after_sync();
    const uint32_t tb = *tmem_slot;
    asm volatile("griddepcontrol.wait;" ::: "memory");   // ---- global memory may be touched from here on ----
#ifdef ESC_TC_TRACE
    TC_TRACE_L(14, launch_id);
#endif
    if (threadIdx.x == 0) TC_TRACE(10, 0);

    // state warps own the carry: row `krow` of the [d_k x 16] slice per thread, fp32 registers
    const bool st_warp = warp >= 12 && warp < 16;
    const bool st_active = st_warp && (DK == 128 || lane < 16);
    const uint32_t krow = (DK == 128) ? 32 * q + lane : 16 * q + (lane & 15);
    float S[16];
    // [S_hi | S_lo] as UMMA B operand, MN-major interleaved: (n,k) -> (n/8)*SBO_S + (k/8)*128 + (k%8)*16 + (n%8)*2,
    // columns n = 0..15 hold the hi terms, 16..31 the lo terms
    auto write_s_operand = [&](uint32_t buf) {
        if (st_active) {
            uint8_t* base = sm + L::s_off + buf * L::s_bytes + (krow >> 3) * 128 + (krow & 7) * 16;
#pragma unroll
            for (int nb = 0; nb < 2; ++nb) {
                uint4 hi, lo;
                hi.x = split2(S[8 * nb + 0], S[8 * nb + 1], lo.x);
                hi.y = split2(S[8 * nb + 2], S[8 * nb + 3], lo.y);
                hi.z = split2(S[8 * nb + 4], S[8 * nb + 5], lo.z);
                hi.w = split2(S[8 * nb + 6], S[8 * nb + 7], lo.w);
                *reinterpret_cast<uint4*>(base + nb * SBO_S) = hi;
                *reinterpret_cast<uint4*>(base + (2 + nb) * SBO_S) = lo;
            }
        }
    };

    if (warp == 0) {
        // ================= TMA producer =================
        if (lane == 0) {
            for (uint32_t c = NS; c < n_chunks && c < (uint32_t)(NS + kPrefetchAhead); ++c) tma_prefetch_chunk(c);
            for (uint32_t c = 0; c < n_chunks; ++c) {
                if (c + NS + kPrefetchAhead < n_chunks) tma_prefetch_chunk(c + NS + kPrefetchAhead);
                // the stage is free once the P, O1 and U issuers of all CS CTAs have committed chunk c - NS (this CTA writes into all
                // of them); O2 reads V from the copy the V~ warps made, so the score path never holds a stage
                mbar_wait_relaxed(&bars[BI.empty + c % NS], ((c / NS) & 1) ^ 1);
                tma_issue(c);
            }
            // tail: every peer's last commits have reached this CTA's barriers before anyone may exit
            for (uint32_t c = n_chunks > (uint32_t)NS ? n_chunks - NS : 0; c < n_chunks; ++c)
                mbar_wait(&bars[BI.empty + c % NS], (c / NS) & 1);
        }
    } else if (warp == 1) {
        // ================= gate warp: b2_i = sum_{r<=i in chunk} log2 g_r, 256 tokens per batch =================
        const uint32_t n_batches = (uint32_t)((T + kGateBatch - 1) / kGateBatch);
        constexpr int GL = C / 8;   // lanes per chunk
        float gv[8];
        auto load_g = [&](uint32_t bt) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const uint64_t tt = (uint64_t)bt * kGateBatch + 8 * lane + u;
                gv[u] = tt < T ? g[((size_t)b * t_stride + tt) * H + h] : 1.f;
            }
        };
        if (n_batches) load_g(0);
        for (uint32_t bt = 0; bt < n_batches; ++bt) {
            float loc[8], run = 0.f;
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                run += log2f(gv[u]);
                loc[u] = run;
            }
            if (bt + 1 < n_batches) load_g(bt + 1);   // next batch's loads fly while this one is scanned
            float incl = run;
#pragma unroll
            for (int d = 1; d < GL; d <<= 1) {
                const float up = __shfl_up_sync(0xffffffffu, incl, d);
                if ((lane % GL) >= d) incl += up;
            }
            const float prev = __shfl_up_sync(0xffffffffu, incl, 1);
            const float excl = (lane % GL) ? prev : 0.f;
            const uint32_t slot = bt & 1;
            mbar_wait_relaxed(&bars[BI.g_empty + slot], ((bt >> 1) & 1) ^ 1);
            float* b2 = gate + slot * 2 * kGateBatch;
            float* eb = b2 + kGateBatch;
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const float x = excl + loc[u];
                b2[8 * lane + u] = x;
                eb[8 * lane + u] = ex2(x);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BI.g_full + slot]);
        }
    } else if (warp == 2) {
        // ================= issuer: P[:, key0 .. key0+NA) = Q K[key0 .. key0+NA)^T =================
        if (lane == 0) {
            constexpr uint32_t idP = idesc_bf16(C, NA, 0, 0);
            // descriptors of stage 0; per chunk / per MMA they are only advanced (the issuing thread's instruction count per
            // MMA is what paces the kernel)
            const uint64_t dQ0 = smem_desc(sm_a + L::stage_off, 16, 1024, kSwz128);
            const uint64_t dK0 = smem_desc(sm_a + L::stage_off + L::q_bytes + key0 * 128, 16, 1024, kSwz128);
            for (uint32_t c = 0; c < n_chunks; ++c) {
                const uint32_t s = c % NS, pb = c % NB;
                mbar_wait(&bars[BI.full + s], (c / NS) & 1);
                mbar_wait(&bars[BI.p_empty + pb], ((c / NB) & 1) ^ 1);
                tc_fence_after_sync();
                const uint64_t dQ = smem_desc_advance(dQ0, s * L::stage_bytes), dK = smem_desc_advance(dK0, s * L::stage_bytes);
                const uint32_t dP = tb + L::tm_p + pb * L::p_cols;
#pragma unroll
                for (int ks = 0; ks < DK / 16; ++ks) {
                    const uint32_t off = (ks / 4) * L::half_bytes + (ks % 4) * 32;
                    mma_bf16_ss(dP, smem_desc_advance(dQ, off), smem_desc_advance(dK, off), idP, ks > 0);
                }
                mma_commit(&bars[BI.p_full + pb]);
                commit_all(&bars[BI.empty + s]);
                TC_TRACE(1, c);
            }
        }
    } else if (warp == 3) {
        // ================= issuer: O1 = Q [S_hi | S_lo] — the only MMA that reads the carried state =================
        if (lane == 0) {
            constexpr uint32_t idO1 = idesc_bf16(C, kTcNM, 0, 1);
            const uint64_t dQ0 = smem_desc(sm_a + L::stage_off, 16, 1024, kSwz128);
            const uint64_t dS0 = smem_desc(sm_a + L::s_off, 128, SBO_S, kSwzNone);
            for (uint32_t c = 0; c < n_chunks; ++c) {
                const uint32_t s = c % NS, ob = c & 1, sb = c % NSB;
                mbar_wait(&bars[BI.full + s], (c / NS) & 1);
                mbar_wait(&bars[BI.o_empty + ob], ((c >> 1) & 1) ^ 1);
                mbar_wait(&bars[BI.s_full + sb], (c / NSB) & 1);
                tc_fence_after_sync();
                TC_TRACE(2, c);
                const uint64_t dQ = smem_desc_advance(dQ0, s * L::stage_bytes), dS = smem_desc_advance(dS0, sb * L::s_bytes);
                const uint32_t dO = tb + L::tm_o1 + ob * 32;
#pragma unroll
                for (int ks = 0; ks < DK / 16; ++ks) {
                    const uint32_t off = (ks / 4) * L::half_bytes + (ks % 4) * 32;
                    mma_bf16_ss(dO, smem_desc_advance(dQ, off), smem_desc_advance(dS, 2 * ks * 128), idO1, ks > 0);
                }
                mma_commit(&bars[BI.s_empty + sb]);
                mma_commit(&bars[BI.o1_full + ob]);
                commit_all(&bars[BI.empty + s]);
            }
        }
    } else if (warp == 4) {
        // ================= issuer: U = K^T [V~_hi | V~_lo] (A operand = the K tile read MN-major) =================
        if (lane == 0) {
            constexpr uint32_t idU = idesc_bf16(DK, kTcNM, 1, 1);
            const uint64_t dK0 = smem_desc(sm_a + L::stage_off + L::q_bytes, L::half_bytes, 1024, kSwz128);
            const uint64_t dV0 = smem_desc(sm_a + L::vt_off, 128, SBO_V, kSwzNone);
            for (uint32_t c = 0; c < n_chunks; ++c) {
                const uint32_t s = c % NS, pb = c % NB, ob = c & 1;
                mbar_wait(&bars[BI.full + s], (c / NS) & 1);
                mbar_wait(&bars[BI.u_empty + ob], ((c >> 1) & 1) ^ 1);
                mbar_wait(&bars[BI.vt_full + pb], (c / NB) & 1);   // the V~ warps are then also done with the stage's V tile
                tc_fence_after_sync();
                TC_TRACE(3, c);
                const uint64_t dK = smem_desc_advance(dK0, s * L::stage_bytes), dV = smem_desc_advance(dV0, pb * L::vt_bytes);
                const uint32_t dU = tb + L::tm_u + ob * 32;
#pragma unroll
                for (int ks = 0; ks < C / 16; ++ks)
                    mma_bf16_ss(dU, smem_desc_advance(dK, 2 * ks * 1024), smem_desc_advance(dV, 2 * ks * 128), idU, ks > 0);
                mma_commit(&bars[BI.u_full + ob]);
                mma_commit(&bars[BI.vt_empty + pb]);
                commit_all(&bars[BI.empty + s]);
            }
        }
    } else if (warp == 5) {
        // ================= issuer: O2 = A_hi V + A_lo V (B operand = the V tile copy, MN-major, 32B swizzle) =================
        if (lane == 0) {
            constexpr uint32_t idO2 = idesc_bf16(C, kTcDVT, 0, 1);
            const uint64_t dA0 = smem_desc(sm_a + L::a_off, L::a_lbo, 128, kSwzNone);
            const uint64_t dV0 = smem_desc(sm_a + L::vt_off + L::vc_off, 512, 256, kSwz32);
            for (uint32_t c = 0; c < n_chunks; ++c) {
                const uint32_t pb = c % NB, ob = c & 1;
                mbar_wait(&bars[BI.o_empty + ob], ((c >> 1) & 1) ^ 1);
                mbar_wait(&bars[BI.vt_full + pb], (c / NB) & 1);   // the V copy
                mbar_wait(&bars[BI.a_full + pb], (c / NB) & 1);    // own slice written + every peer's slice landed
                tc_fence_after_sync();
                TC_TRACE(4, c);
                const uint64_t dA = smem_desc_advance(dA0, pb * L::a_bytes), dV = smem_desc_advance(dV0, pb * L::vt_bytes);
                const uint32_t dO = tb + L::tm_o2 + ob * 16;
#pragma unroll
                for (int term = 0; term < 2; ++term) {
#pragma unroll
                    for (int ks = 0; ks < C / 16; ++ks)
                        mma_bf16_ss(dO, smem_desc_advance(dA, term * L::a_term + 2 * ks * L::a_lbo), smem_desc_advance(dV, 2 * ks * 256), idO2,
                                    (term | ks) > 0);
                }
                mma_commit(&bars[BI.o2_full + ob]);
                mma_commit(&bars[BI.vt_empty + pb]);
                commit_all(&bars[BI.a_empty + pb]);   // every CTA writes into this buffer: all of them must know
            }
        }
    } else if (warp == 6 || warp == 7 || warp == 20 || warp == 21) {
        // ================= V~ warps: [V~_hi | V~_lo], V~_j = 2^(b_C - b_j) v_j, and a copy of V for O2 =================
        // UMMA B operand, MN-major interleaved: (n,k=token) -> (n/8)*SBO_V + (k/8)*128 + (k%8)*16 + (n%8)*2
        const int tid_v = (warp < 8 ? warp - 6 : warp - 18) * 32 + lane;
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t s = c % NS, pb = c % NB, bt = c / CPB, gslot = bt & 1;
            mbar_wait(&bars[BI.g_full + gslot], (bt >> 1) & 1);
            const float* b2 = gate + gslot * 2 * kGateBatch + (c % CPB) * C;
            mbar_wait(&bars[BI.full + s], (c / NS) & 1);
            mbar_wait(&bars[BI.vt_empty + pb], ((c / NB) & 1) ^ 1);
            const uint8_t* vs = sm + L::stage_off + s * L::stage_bytes + 2 * L::q_bytes;
            uint8_t* vt = sm + L::vt_off + pb * L::vt_bytes;
            const float b_last = b2[C - 1];
#pragma unroll
            for (int it = 0; it < 2 * C / kVtThreads; ++it) {
                const int idx = tid_v + it * kVtThreads, j = idx >> 1, half = idx & 1;
                const uint32_t voff = j * 32 + ((half ^ ((j >> 2) & 1)) * 16);   // undo 32B swizzle
                const uint4 raw = *reinterpret_cast<const uint4*>(vs + voff);
                *reinterpret_cast<uint4*>(vt + L::vc_off + voff) = raw;          // the V tile itself, same (swizzled) placement: O2's operand
                const float sc = ex2(b_last - b2[j]);
                const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
                uint32_t hi[4], lo[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float x0 = __uint_as_float(w[e] << 16) * sc, x1 = __uint_as_float(w[e] & 0xFFFF0000u) * sc;
                    hi[e] = split2(x0, x1, lo[e]);
                }
                const uint32_t off = half * SBO_V + (j >> 3) * 128 + (j & 7) * 16;
                *reinterpret_cast<uint4*>(vt + off) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                *reinterpret_cast<uint4*>(vt + 2 * SBO_V + off) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
            }
            fence_proxy_async_smem();   // generic-proxy writes -> visible to tcgen05.mma's operand reads
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bars[BI.vt_full + pb]);
                if ((c % CPB) == (uint32_t)CPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
            }
        }
    }
    else if ((warp >= 8 && warp < 12) || warp >= kTcWarps) {
        // ================= score warps: A[:, slice] = P[:, slice] ⊙ 2^(b_i - b_j) (causal) -> every CTA of the cluster =================
        // One warp per TMEM lane quadrant.  A quadrant holds 16 rows of an M = 64 tile (row r in lane 32(r/16) + r%16) or 32
        // rows of an M = 128 tile (row r in lane r): NG 16-row groups per warp.  A group whose rows all precede the slice's
        // first key is entirely above the diagonal: it is skipped here and never written anywhere (it stays zero).
        constexpr int NG = C / 64;
        constexpr uint32_t kSlice = (NA / 8) * L::a_lbo;           // bytes of one CTA's slice
        constexpr uint32_t tx = (CS - 1) * kSlice;                  // what the peers push into this CTA's A buffer per chunk
        auto rows_base = [&](int qq, int gi) { return (C == 64) ? 16 * qq : 32 * qq + 16 * gi; };
        const uint32_t kw0 = key0 + (warp >= kTcWarps ? NAW : 0);   // first key column of this warp
        bool act[NG];   // (a CTA on its own writes all of A itself: masked groups as zeros)
#pragma unroll
        for (int gi = 0; gi < NG; ++gi) act[gi] = CS == 1 || (uint32_t)rows_base(q, gi) + 15 >= key0;
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t pb = c % NB, bt = c / CPB, gslot = bt & 1;
            mbar_wait(&bars[BI.g_full + gslot], (bt >> 1) & 1);
            const float* b2 = gate + gslot * 2 * kGateBatch + (c % CPB) * C;
            if (q == 3 && lane == 0) TC_TRACE(5, c);
            // every b_j is read before the first A store (the stores may alias b2 as far as the compiler can tell)
            float2 bj[NAW / 8];
#pragma unroll
            for (int jb = 0; jb < NAW / 8; ++jb) bj[jb] = *reinterpret_cast<const float2*>(b2 + kw0 + jb * 8 + 2 * (lane & 3));
            float bi[NG][2];
#pragma unroll
            for (int gi = 0; gi < NG; ++gi) {
                bi[gi][0] = b2[rows_base(q, gi) + (lane >> 2)];
                bi[gi][1] = b2[rows_base(q, gi) + (lane >> 2) + 8];
            }
            mbar_wait(&bars[BI.a_empty + pb], ((c / NB) & 1) ^ 1);   // all CS CTAs are done reading A buffer pb (chunk c - NB)
            mbar_wait(&bars[BI.p_full + pb], (c / NB) & 1);
            tc_fence_after_sync();
            uint32_t r[NG][NAW / 2];
#pragma unroll
            for (int gi = 0; gi < NG; ++gi)
                if (act[gi])
                    tmem_ld_slice<NAW>(tmem_addr(tb, (C == 64) ? 32 * q : 32 * q + 16 * gi, L::tm_p + pb * L::p_cols + (kw0 - key0)), r[gi]);
            tmem_ld_wait();
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BI.p_empty + pb]);   // this warp's part of P(c) is in registers
            uint8_t* ab = sm + L::a_off + pb * L::a_bytes;
#pragma unroll
            for (int gi = 0; gi < NG; ++gi) {
                if (act[gi]) {
                    const int ra = rows_base(q, gi) + (lane >> 2), rb = ra + 8;
                    uint32_t hi_a[NAW / 8], lo_a[NAW / 8], hi_c[NAW / 8], lo_c[NAW / 8];
#pragma unroll
                    for (int jb = 0; jb < NAW / 8; ++jb) {
                        const int j0 = (int)kw0 + jb * 8 + 2 * (lane & 3);
                        float a0 = __uint_as_float(r[gi][4 * jb + 0]) * ex2(bi[gi][0] - bj[jb].x);
                        float a1 = __uint_as_float(r[gi][4 * jb + 1]) * ex2(bi[gi][0] - bj[jb].y);
                        float c0 = __uint_as_float(r[gi][4 * jb + 2]) * ex2(bi[gi][1] - bj[jb].x);
                        float c1 = __uint_as_float(r[gi][4 * jb + 3]) * ex2(bi[gi][1] - bj[jb].y);
                        a0 = (j0 <= ra) ? a0 : 0.f;       // causal mask j <= i
                        a1 = (j0 + 1 <= ra) ? a1 : 0.f;
                        c0 = (j0 <= rb) ? c0 : 0.f;
                        c1 = (j0 + 1 <= rb) ? c1 : 0.f;
                        hi_a[jb] = split2(a0, a1, lo_a[jb]);
                        hi_c[jb] = split2(c0, c1, lo_c[jb]);
                    }
                    uint8_t* arow = ab + (ra >> 3) * 128 + (ra & 7) * 16 + (lane & 3) * 4;
#pragma unroll
                    for (int jb = 0; jb < NAW / 8; ++jb) {
                        uint8_t* pa = arow + (kw0 / 8 + jb) * L::a_lbo;
                        *reinterpret_cast<uint32_t*>(pa) = hi_a[jb];
                        *reinterpret_cast<uint32_t*>(pa + L::a_term) = lo_a[jb];
                        *reinterpret_cast<uint32_t*>(pa + 128) = hi_c[jb];              // row + 8
                        *reinterpret_cast<uint32_t*>(pa + 128 + L::a_term) = lo_c[jb];
                    }
                }
            }
            fence_proxy_async_smem();   // generic-proxy writes of A -> visible to the bulk copies and to tcgen05.mma
            __syncwarp();
            // the slice of this CTA (all rows, both terms: NA/8 consecutive 8-key groups) is one contiguous range of the A
            // buffer: once the four score warps have written it, one lane per peer pushes it into the same place of that
            // peer's buffer pb; the copy completes (tx bytes) on the peer's a_full barrier
            if constexpr (CS > 1) {   // (on its own a CTA has nobody to push to)
                if constexpr (SW == 1) asm volatile("bar.sync 1, 128;" ::: "memory");
                else asm volatile("bar.sync 1, 256;" ::: "memory");
            }
            if constexpr (CS > 1) if (q == 0 && warp < kTcWarps && lane + 1 < CS) {
                const uint32_t d = (uint32_t)lane + ((uint32_t)lane >= rank ? 1u : 0u);
                const uint32_t off = L::a_off + pb * L::a_bytes + (key0 / 8) * L::a_lbo;
                bulk_copy_to_cluster(mapa(sm_a + off, d), sm_a + off, kSlice, mapa(smem_u32(&bars[BI.a_full + pb]), d));
            }
            if (q == 3 && lane == 0) TC_TRACE(6, c);
            if (lane == 0) {
                if (CS > 1 && q == 3 && warp < kTcWarps) mbar_arrive_expect_tx(&bars[BI.a_full + pb], tx);   // quadrant 3 holds the last rows: always active
                else mbar_arrive(&bars[BI.a_full + pb]);
                if ((c % CPB) == (uint32_t)CPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
            }
        }
        // tail: the peers' last O2 commits have reached this CTA's barriers before anyone may exit
        for (uint32_t c = n_chunks > (uint32_t)NB ? n_chunks - NB : 0; c < n_chunks; ++c)
            mbar_wait(&bars[BI.a_empty + c % NB], (c / NB) & 1);
    } else if (st_warp) {
        // ================= state warps: the carry  S <- 2^(b_C) S + (Uh + Ul), fp32 FMA in registers =================
#pragma unroll
        for (int j = 0; j < 16; ++j) S[j] = 0.f;
        if (st_active && state_in) {
            const float4* p = reinterpret_cast<const float4*>(state_in + ((size_t)bh * DK + krow) * DV + dv0);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float4 x = p[j];
                S[4 * j] = x.x; S[4 * j + 1] = x.y; S[4 * j + 2] = x.z; S[4 * j + 3] = x.w;
            }
        }
        write_s_operand(0);   // version 0 of the S operand (read by O1(0))
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars[BI.s_full]);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t ob = c & 1, bt = c / CPB, gslot = bt & 1;
            mbar_wait(&bars[BI.g_full + gslot], (bt >> 1) & 1);
            const float gam = gate[gslot * 2 * kGateBatch + kGateBatch + (c % CPB) * C + C - 1];
            mbar_wait(&bars[BI.u_full + ob], (c >> 1) & 1);
            tc_fence_after_sync();
            uint32_t ur[32];
            tmem_ld_32x32b_x32(tmem_addr(tb, 32 * q, L::tm_u + ob * 32), ur);
            tmem_ld_wait();
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bars[BI.u_empty + ob]);
                if ((c % CPB) == CPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
            }
#pragma unroll
            for (int j = 0; j < 16; ++j) S[j] = fmaf(gam, S[j], __uint_as_float(ur[j]) + __uint_as_float(ur[16 + j]));
            if (c + 1 < n_chunks) {   // version c+1 of the S operand (read by O1(c+1))
                const uint32_t sb = (c + 1) % NSB;
                mbar_wait(&bars[BI.s_empty + sb], ((((c + 1) / NSB) & 1) ^ 1));
                write_s_operand(sb);
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars[BI.s_full + sb]);
            }
            if (q == 3 && lane == 0) TC_TRACE(7, c);
        }
        if (st_active) {
            float4* p = reinterpret_cast<float4*>(state_out + ((size_t)bh * DK + krow) * DV + dv0);
#pragma unroll
            for (int j = 0; j < 4; ++j) p[j] = make_float4(S[4 * j], S[4 * j + 1], S[4 * j + 2], S[4 * j + 3]);
        }
    } else if (warp >= 16 && warp < 20) {
        // ================= epilogue warps: o_i = 2^(b_i) (O1h_i + O1l_i) + O2_i =================
        constexpr int NG = C / 64;
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t ob = c & 1, bt = c / CPB, gslot = bt & 1;
            mbar_wait(&bars[BI.g_full + gslot], (bt >> 1) & 1);
            const float* eb = gate + gslot * 2 * kGateBatch + kGateBatch + (c % CPB) * C;
            mbar_wait_relaxed(&bars[BI.o2_full + ob], (c >> 1) & 1);
            mbar_wait_relaxed(&bars[BI.o1_full + ob], (c >> 1) & 1);
            tc_fence_after_sync();
            const uint64_t t0 = (uint64_t)c * C;
            const int n = (int)((T - t0) < (uint64_t)C ? (T - t0) : (uint64_t)C);
#pragma unroll
            for (int gi = 0; gi < NG; ++gi) {
                const int rg = (C == 64) ? q : 2 * q + gi;
                const uint32_t lane_base = (C == 64) ? 32 * q : 32 * q + 16 * gi;
                uint32_t r1[16], r2[8];
                tmem_ld_16x256b_x4(tmem_addr(tb, lane_base, L::tm_o1 + ob * 32), r1);
                tmem_ld_16x256b_x2(tmem_addr(tb, lane_base, L::tm_o2 + ob * 16), r2);
                tmem_ld_wait();
                const int ra = 16 * rg + (lane >> 2), rb = ra + 8;
                const float ea = eb[ra], ebb = eb[rb];
                if (gi == NG - 1) {
                    tc_fence_before_sync();
                    __syncwarp();
                    if (lane == 0) {
                        mbar_arrive(&bars[BI.o_empty + ob]);
                        if ((c % CPB) == CPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
                    }
                }
                OutT* oa = o + (((size_t)b * t_stride + t0 + ra) * H + h) * DV + dv0 + 2 * (lane & 3);
                OutT* oc = o + (((size_t)b * t_stride + t0 + rb) * H + h) * DV + dv0 + 2 * (lane & 3);
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {   // columns 8 jb + 2(t%4) + {0,1}: hi terms in block jb, lo terms in block 2 + jb
                    const float h0 = __uint_as_float(r1[4 * jb + 0]) + __uint_as_float(r1[4 * (2 + jb) + 0]);
                    const float h1 = __uint_as_float(r1[4 * jb + 1]) + __uint_as_float(r1[4 * (2 + jb) + 1]);
                    const float h2 = __uint_as_float(r1[4 * jb + 2]) + __uint_as_float(r1[4 * (2 + jb) + 2]);
                    const float h3 = __uint_as_float(r1[4 * jb + 3]) + __uint_as_float(r1[4 * (2 + jb) + 3]);
                    if (ra < n) store_o2<OutT>(oa + jb * 8, fmaf(ea, h0, __uint_as_float(r2[4 * jb + 0])), fmaf(ea, h1, __uint_as_float(r2[4 * jb + 1])));
                    if (rb < n) store_o2<OutT>(oc + jb * 8, fmaf(ebb, h2, __uint_as_float(r2[4 * jb + 2])), fmaf(ebb, h3, __uint_as_float(r2[4 * jb + 3])));
                }
            }
            if (q == 3 && lane == 0) TC_TRACE(8, c);
        }
    }

    // ---- teardown: every tcgen05 op of this CTA has completed (the state and epilogue warps waited on the last commits),
    // and no peer still multicasts, copies or arrives into this CTA once the whole cluster is here ----
    tc_fence_before_sync();
    if (threadIdx.x == 0) TC_TRACE(11, 0);
    if constexpr (CS > 1) cluster_sync_relaxed();
    else __syncthreads();
    if (threadIdx.x == 0) TC_TRACE(12, 0);
#ifdef ESC_TC_TRACE
    TC_TRACE_L(15, launch_id);
#endif
    if (warp == 2) tmem_dealloc(tb, L::tmem_cols);
}

// ---- host ---------------------------------------------------------------------------------------
typedef CUresult (*TmapEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static TmapEncodeFn tmap_encode_fn() {
    static TmapEncodeFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess)
            p = nullptr;
        return (TmapEncodeFn)p;
    }();
    return fn;
}

// 4-D map over a [B, t_stride, H, D] bf16 tensor whose first `T` tokens per batch row are valid:
// dims (D, H, T, B), box (box_d, 1, box_t, 1).  Rows beyond T read as zero (the short last chunk).
static int make_tmap(CUtensorMap* m, const void* base, uint32_t D, uint32_t H, uint64_t T, uint64_t t_stride, uint32_t B,
                     uint32_t box_d, uint32_t box_t, CUtensorMapSwizzle sw) {
    TmapEncodeFn enc = tmap_encode_fn();
    if (!enc) return ESC_ERR_CUDA;
    cuuint64_t dims[4] = {D, H, T ? T : 1, B};
    cuuint64_t strides[3] = {(cuuint64_t)D * 2, (cuuint64_t)H * D * 2, (cuuint64_t)t_stride * H * D * 2};
    cuuint32_t box[4] = {box_d, 1, box_t, 1};
    cuuint32_t es[4] = {1, 1, 1, 1};
    if (B == 1) strides[2] = strides[1] * dims[2];   // unused dimension: any valid multiple of 16
    CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, es,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? ESC_OK : ESC_ERR_CUDA;
}

// whole Q / K tiles for the cluster-free variant: dimensions (d % 64, t, d / 64, h, b), box (64, box_t, D / 64, 1, 1)
static int make_tmap_halves(CUtensorMap* m, const void* base, uint32_t D, uint32_t H, uint64_t T, uint64_t t_stride, uint32_t B,
                            uint32_t box_t) {
    TmapEncodeFn enc = tmap_encode_fn();
    if (!enc) return ESC_ERR_CUDA;
    const uint32_t nh = D / 64;
    cuuint64_t dims[5] = {64, T ? T : 1, nh, H, B};
    cuuint64_t strides[4] = {(cuuint64_t)H * D * 2, 128, (cuuint64_t)D * 2, (cuuint64_t)t_stride * H * D * 2};
    cuuint32_t box[5] = {64, box_t, nh, 1, 1};
    cuuint32_t es[5] = {1, 1, 1, 1, 1};
    if (B == 1) strides[3] = strides[0] * dims[1];   // unused dimension: any valid multiple of 16
    CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void*>(base), dims, strides, box, es,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? ESC_OK : ESC_ERR_CUDA;
}

template <int DK, int C, int CS, typename OutT>
static int launch_tc_t(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* state_in,
                       float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    using L = TcCfg<DK, C, CS>;
    constexpr uint32_t slot = kSlotScan + (DK == 128 ? 0 : 1) + 2 * (CS > 1 ? 1 : 0) + 4 * (sizeof(OutT) == 4 ? 0 : 1);
    {
        const int rc = ensure_dyn_smem(ctx, slot, esc_scan_tc_kernel<DK, C, CS, OutT>, (int)L::total);
        if (rc != ESC_OK) return rc;
    }
    if (!state_out) return ESC_OK;   // prepare-only call (before a stream capture)
    CUtensorMap tq, tk, tv;
    const void* qq = T ? q : (const void*)state_out;   // T == 0: maps are never dereferenced, any valid address will do
    const void* kk = T ? k : (const void*)state_out;
    const void* vv = T ? v : (const void*)state_out;
    // Q / K: each CTA of the cluster loads (and multicasts) C / CS rows of a chunk; V: the CTA's own 16 columns
    int rc;
    if (CS == 1) {
        rc = make_tmap_halves(&tq, qq, DK, s.H, T, t_stride ? t_stride : 1, s.B, C);
        if (rc == ESC_OK) rc = make_tmap_halves(&tk, kk, DK, s.H, T, t_stride ? t_stride : 1, s.B, C);
    } else {
        rc = make_tmap(&tq, qq, DK, s.H, T, t_stride ? t_stride : 1, s.B, 64, C / CS, CU_TENSOR_MAP_SWIZZLE_128B);
        if (rc == ESC_OK) rc = make_tmap(&tk, kk, DK, s.H, T, t_stride ? t_stride : 1, s.B, 64, C / CS, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (rc == ESC_OK) rc = make_tmap(&tv, vv, s.dv, s.H, T, t_stride ? t_stride : 1, s.B, kTcDVT, C, CU_TENSOR_MAP_SWIZZLE_32B);
    if (rc != ESC_OK) return rc;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(s.dv / kTcDVT, s.B * s.H);   // d_v / 16 CTAs per (b, h), in clusters of CS
    cfg.blockDim = dim3(TcScore<CS>::threads);
    cfg.dynamicSmemBytes = L::total;
    cfg.stream = stream;
    cudaLaunchAttribute attr[2];
    memset(attr, 0, sizeof attr);   // the value union is wider than the fields set below; stale stack bytes there changed the kernel time by 9 % (r01)
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddepcontrol.* in the kernel
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = CS;
    attr[1].val.clusterDim.y = 1;
    attr[1].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = CS > 1 ? 2 : 1;
    ESC_CUDA(cudaLaunchKernelEx(&cfg, esc_scan_tc_kernel<DK, C, CS, OutT>, tq, tk, tv, g, state_in, state_out, (OutT*)o, s.H, s.dv, T,
                                t_stride));
    return ESC_OK;
}

template <int DK, int C, int CS>
static int launch_tc_o(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* state_in,
                       float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    if (s.out_dtype == ESC_DTYPE_F32) return launch_tc_t<DK, C, CS, float>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    return launch_tc_t<DK, C, CS, bf16>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
}

// Cluster size: 4.  A cluster of 8 (all d_v slices of a d_v = 128 head) would share twice as much, but B200 can keep only 15
// such clusters resident at this shared-memory footprint (cudaOccupancyMaxActiveClusters, r01): the 16 heads of the B = 1
// workloads would run as two waves.  Clusters of 4 fit 33 times: 32 clusters (128 CTAs) in one wave.
constexpr int kTcCluster = 4;
// Short calls (the suffix scan after a restore: one or two chunks) run WITHOUT a cluster: every CTA loads whole Q / K tiles
// and computes all C columns of P and A itself.  Per chunk that is 4x the score arithmetic and 4x the L2 -> SM traffic, but
// a one-chunk call is a single pass through the dependent pipeline, and dropping the slice exchange and both cluster barriers
// from it is worth more (r01, 18-layer suffix graph: 5.35 -> 4.78 us per layer at T = 64, 6.54 -> 6.20 at 128, 8.25 -> 8.48
// at 256).  Same MMAs in the same order on the same operands: the results are bit-identical to the cluster variant's
// (tests: restore + short suffix against the cold run).
#ifndef ESC_TC_SHORT
#define ESC_TC_SHORT 128
#endif
constexpr uint64_t kTcShortT = ESC_TC_SHORT;

template <int DK, int C>
static int launch_tc_dv(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* state_in,
                        float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    if (s.dv % (kTcDVT * kTcCluster)) return ESC_ERR_UNSUPPORTED;
    if (!state_out) {   // prepare-only call: both variants
        const int rc = launch_tc_o<DK, C, 1>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
        if (rc != ESC_OK) return rc;
    } else if (T <= kTcShortT) {
        return launch_tc_o<DK, C, 1>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    }
    return launch_tc_o<DK, C, kTcCluster>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
}

// The key's chunk (64 or 128) is the alignment grid the caller commits to (restore boundaries are multiples of it); the
// kernel's token tile is 64 for both: the recurrence is the same function, a 128-aligned boundary is also 64-aligned (so
// restore + continue stays bit-identical to the cold run), and the 64-token tile is 2.1x faster than a 128-token one
// (r01 sweep: 83 M vs 38 M tokens/s at T = 64k — A grows quadratically with the tile and leaves no room for buffering).
// The kernel template stays generic in C (the 128-token instantiation passed the same parity tests before this change).
int launch_scan_tc(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* state_in,
                   float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    if (s.chunk != 64 && s.chunk != 128) return ESC_ERR_UNSUPPORTED;
    if (s.dk == 128) return launch_tc_dv<128, 64>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    if (s.dk == 64) return launch_tc_dv<64, 64>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    return ESC_ERR_UNSUPPORTED;
}

#ifdef ESC_TC_TRACE
extern "C" int esc_debug_trace_read(long long* host) {
    return (int)cudaMemcpyFromSymbol(host, g_tc_trace, sizeof(g_tc_trace));
}
extern "C" int esc_debug_max_clusters(int* out8, int* out4) {
    using L = TcCfg<128, 64, 4>;
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3(kTcThreads);
    cfg.dynamicSmemBytes = L::total;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaFuncSetAttribute(esc_scan_tc_kernel<128, 64, 4, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::total);
    cudaFuncSetAttribute(esc_scan_tc_kernel<128, 64, 4, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::total);
    attr[0].val.clusterDim.x = 4; cfg.gridDim = dim3(8, 64);
    cudaError_t e = cudaOccupancyMaxActiveClusters(out8, esc_scan_tc_kernel<128, 64, 4, float>, &cfg);
    attr[0].val.clusterDim.x = 4; cfg.gridDim = dim3(4, 64);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveClusters(out4, esc_scan_tc_kernel<128, 64, 4, float>, &cfg);
    return (int)e;
}
#endif

}  // namespace esc
