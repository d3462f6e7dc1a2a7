// Gated delta-rule scan, chunked (WY) form on tcgen05 / TMEM / TMA, 64-token chunks (include/esc.h: esc_gdn_scan).
//
//     u_t = k_t (a_t S_{t-1}) ,  S_t = a_t S_{t-1} + beta_t k_t^T (v_t - u_t) ,  o_t = q_t S_t
//
// Per chunk of C = 64 tokens, S the state at the chunk's start, b_i = sum_{r<=i} log2 a_r (inclusive, inside the chunk),
// D_ij = 2^(b_i - b_j) (<= 1 for j <= i), Gamma = diag(2^(b_i)), w_i = beta_i (v_i - u_i) the rows the 64 rank-one updates add:
//     G = K K^T , P = Q K^T                                   (64 x 64)    tcgen05.mma  M=64 N=64 K=d_k   (SS); G in the owning CTA only
//     A^k_ij = beta_i D_ij G_ij  (j <  i) ,  T = (I + A^k)^-1  (64 x 64)    fp32 ALU + warp-level MMAs, OFF the carry chain
//     A^q_ij =        D_ij P_ij  (j <= i)                      (64 x 64)    in place in TMEM (bf16 hi | lo), as in scan_kernel.cu
//     [X | Y] = [K ; Q] [S_hi | S_lo]                          (64 x 2W)    tcgen05.mma  M=64 N=2W K=d_k   (SS), W = 16 columns
//     R = beta (.) (V - Gamma X)                               (64 x W)     fp32, registers
//     Wm = T R = T_hi [R_hi | R_lo] + T_lo R_hi                (64 x W)     tcgen05.mma  M=64 K=64         (SS)   (w_i = row i of Wm)
//     o = Gamma Y + A^q_hi [Wm_hi | Wm_lo] + A^q_lo Wm_hi      (64 x W)     tcgen05.mma  M=64 K=64         (TS: A^q from TMEM)
//     U = K^T [W~_hi | W~_lo] , W~_j = 2^(b_C - b_j) Wm_j      (d_k x 2W)   tcgen05.mma  M=d_k K=64        (SS)
//     S_next = 2^(b_C) S + (Uh + Ul)                           fp32 FMA in registers (the carry)
// (substituting w_j for the updates of tokens j < i in u_i = k_i a_i S_{i-1} gives (I + A^k) Wm = R: the chunk's 64
// sequential updates become one unit-lower-triangular system; its inverse depends on k, beta, a only.)
//
// Decomposition: the columns of S are independent, one CTA owns (b, h, 16 columns of d_v) and walks the chunks in order with its
// [d_k x 16] state slice in registers.  The carry chain of a chunk is  S -> X (MMA) -> R (registers) -> Wm (MMA) -> W~
// (registers) -> U (MMA) -> S: three small MMA groups and three register passes; everything else (P, the scores, Y, the
// outputs) is computed beside it by warps of its own and meets the chain through mbarriers.
//
// The inverse T is shared.  T = (I + A^k)^-1 depends on k, beta and the decays only: it is the same matrix in every d_v slice of a
// head.  Four slices form a thread-block cluster, and CTA c % 4 computes T(c) for all of them ("owns" chunk c): its four T warps
// work on one chunk in four, several chunks ahead of the carry chain, with a pipeline of their own (their own gate values, their
// own TMA load of the K tile, G = K K^T issued by themselves), stage the result in shared memory, and a push warp copies it
// into operand slot c % 2 of EVERY CTA of the cluster (cp.async.bulk over distributed shared memory, completion as transaction
// bytes on each CTA's t_full barrier).  Flow control is two remote arrivals per chunk and CTA, from a warp of its own ("my
// Wm(c) has read its copy": the slot is free for T(c + 2), and the owner's staging buffer for its next chunk).
// (I + A^k) is unit lower triangular, 4 x 4 blocks of 16 x 16: each T warp inverts one diagonal block in fp32 (one column per
// lane, forward substitution), then warp J fills block COLUMN J of T by the block recursion
//     T_IJ = - T_II  sum_{K=J}^{I-1} A^k_IK T_KJ      evaluated on the transpose, U = T^T:  U_JI = -(sum_K U_JK (A^k_IK)^T) U_II,
// where the running blocks U_JK are A operands of the next product.  These 16 x 16 x 16 products run as warp-level mma.sync
// (two-term bf16 splits): the only mma.sync in the library, 96 instructions per owned chunk.  The same products in fp32 on the
// CUDA cores (packed FFMA2, two levels of 2 x 2 block inverses, no mma.sync at all) are bit-for-bit as good and were measured
// at 0.410 ms against 0.395 ms for 16 448 tokens: their instruction stream competes with the chain's warps for issue slots.
//
// Warp roles (28 warps, mbarrier pipeline, no CTA-wide barrier in the loop):
//   warp 0       TMA producer (Q, K whole tiles through the 5-D halves map, V tile; L2 prefetch ahead)
//   warp 1       gate warp: b = prefix sums of log2 a, 2^b, beta, 256 tokens per batch
//   warp 2       issuer of P                  warp 3   issuer of the chain (X, Y, Wm, U) and of O2
//   warp 4       ack warp (remote arrivals)   warp 5   push warp (T of an owned chunk -> the cluster)
//   warps 8-11   T warps (the inverse)        warps 12-15  R / W warps (the register passes of the chain)
//   warps 16-19  score warps (A^q in TMEM)    warps 20-23  epilogue (o)            warps 24-27  state warps (the carry)
//
// Bit-identity: a chunk's results are a pure function of (S bits, the chunk's inputs): fixed tile, no atomics,
// no split-K, every accumulator produced by one issuer in a fixed order.  A restore + continue at a boundary that is a multiple
// of 64 tokens from the start of the sequence of calls replays the same chunks: same bits as the cold run.
#include <cuda.h>
#include <string.h>
#include <cuda_bf16.h>

#include "esc_internal.h"
#include "sm100_ptx.cuh"
#include "tmap.h"

namespace esc {

using namespace ptx;

constexpr int kGC = 64;            // tokens per chunk
constexpr int kGW = 16;            // d_v columns per CTA
constexpr int kGBatch = 256;       // tokens per gate batch
constexpr int kGCPB = kGBatch / kGC;
#ifndef ESC_GDN_CLUSTER
#define ESC_GDN_CLUSTER 4
#endif
constexpr int kGdnCluster = ESC_GDN_CLUSTER;   // d_v slices of a head that share the chunk inverses (even)
// Calls of up to kGdnShortT tokens (the suffix after a restore: one chunk) launch WITHOUT the cluster: every CTA inverts its
// own chunks (the same instructions on the same inputs: same bits) and the push is a local copy; with a single chunk there is
// nothing to share, and the cluster launch and the distributed-shared-memory hop are on the first chunk's path.
constexpr uint64_t kGdnShortT = 64;     // (two chunks: 11.3 us without the cluster against 10.9 with it)
constexpr int kGAhead = 4;         // chunks prefetched into L2 ahead of the shared-memory ring

#ifdef ESC_GDN_PROF   // bring-up only: cycles every role of CTA (0,0) spends in each of its waits / sections, and in its loop in total
__device__ long long g_gdn_prof[32 * 8];
#define GPROF_DECL long long prof_[8] = {0, 0, 0, 0, 0, 0, 0, 0}; const long long prof_t0_ = clock64();
#define GW_(slot, call) do { const long long t_ = clock64(); call; prof_[slot] += clock64() - t_; } while (0)
#define GSEG_START long long seg_t_ = clock64();
#define GSEG(slot) do { const long long n_ = clock64(); prof_[slot] += n_ - seg_t_; seg_t_ = n_; } while (0)
#define GPROF_END do { if (blockIdx.x == 0 && blockIdx.y == 0 && lane == 0) { prof_[7] = clock64() - prof_t0_; \
        for (int i_ = 0; i_ < 8; ++i_) g_gdn_prof[warp * 8 + i_] = prof_[i_]; } } while (0)
#else
#define GPROF_DECL
#define GW_(slot, call) call
#define GSEG_START
#define GSEG(slot) do { } while (0)
#define GPROF_END do { } while (0)
#endif

template <int DK>
struct GdnCfg {
    static constexpr int NH = DK / 64;                       // 64-column halves of a Q / K tile
    static constexpr int NS = 3;                             // Q | K stages (2: 4 % slower)
    static constexpr int NV = 4;                             // V tiles
    static constexpr int kWarps = 28;
    static constexpr int kThreads = kWarps * 32;
    static constexpr uint32_t half_bytes = kGC * 128;        // one [64 x 64] bf16 half tile
    static constexpr uint32_t q_bytes = NH * half_bytes;
    static constexpr uint32_t stage_bytes = 2 * q_bytes;     // [Q halves][K halves]
    static constexpr uint32_t s_half_bytes = 2 * kGW * 128;  // S^T operand: rows [S_hi^T (16) | S_lo^T (16)] x 64 columns of d_k, K-major, 128B swizzle
    static constexpr uint32_t s_bytes = NH * s_half_bytes;
    static constexpr uint32_t v_bytes = kGC * kGW * 2;       // [64 x 16] bf16, 32-byte swizzle
    static constexpr uint32_t op_sbo = (kGC / 8) * 128;      // MN-major interleaved operands: (n, k) -> (n/8) op_sbo + (k/8) 128 + (k%8) 16 + (n%8) 2
    static constexpr uint32_t op_bytes = (2 * kGW / 8) * op_sbo;   // [x_hi | x_lo] 64 tokens x 32 columns: R, Wm, W~
    static constexpr uint32_t t_term_bytes = (kGC / 8) * op_sbo;   // T: 64 x 64, one term
    static constexpr uint32_t t_bytes = 2 * t_term_bytes;
    static constexpr uint32_t a_pitch = 144;                 // A^k | U staging matrix: row-major bf16, padded rows (conflict-free ldmatrix)
    static constexpr uint32_t a_term_bytes = kGC * a_pitch;
    static constexpr uint32_t lt_pitch = 20;                 // fp32 diagonal blocks, transposed: LT[j][i]
    static constexpr uint32_t lt_bytes = 4 * 16 * lt_pitch * 4;
    static constexpr uint32_t tg_bytes = 4 * 2 * kGC * 4;      // the T warps' own gate values of a chunk: per warp [b2[64], beta[64]]

    static constexpr uint32_t stage_off = 0;
    static constexpr uint32_t s_off = stage_off + NS * stage_bytes;
    static constexpr uint32_t v_off = s_off + 2 * s_bytes;
    static constexpr uint32_t t_off = v_off + NV * v_bytes;
    static constexpr uint32_t tstage_off = t_off + 2 * t_bytes;   // the T of an owned chunk, before it is pushed to the cluster
    static constexpr uint32_t a_off = tstage_off + t_bytes;       // staging matrix [hi][lo]; first the K tile of the owned chunk (G = K K^T)
    static constexpr uint32_t r_off = a_off + 2 * a_term_bytes;
    static constexpr uint32_t wv_off = r_off + op_bytes;     // [2]
    static constexpr uint32_t wt_off = wv_off + 2 * op_bytes;
    static constexpr uint32_t lt_off = wt_off + op_bytes;
    static constexpr uint32_t tg_off = lt_off + lt_bytes;
    static constexpr uint32_t traw_off = tg_off + tg_bytes;  // [2][a[64], beta[64]] fp32: raw gate inputs of the owned chunks (cp.async, one ahead)
    static constexpr uint32_t gate_off = traw_off + 2 * 2 * kGC * 4;  // [2][b2[256], eb[256], beta[256]] fp32
    static constexpr uint32_t raw_off = gate_off + 2 * 3 * kGBatch * 4;   // [2][a[256], beta[256]] fp32: the gate warp's staging
    static constexpr uint32_t bar_off = raw_off + 2 * 2 * kGBatch * 4;
    static constexpr uint32_t total = bar_off + 64 * 8 + 16 + 1024;
    // TMEM columns
    static constexpr uint32_t tm_p = 0;        // [2] x 64: P -> A^q hi | lo
    static constexpr uint32_t tm_g = 128;      // 64: G of the chunk this CTA inverts (192..255 unused)
    static constexpr uint32_t tm_x = 256;      // 32: X hi | lo
    static constexpr uint32_t tm_y = 288;      // [2] x 32: Y hi | lo
    static constexpr uint32_t tm_w = 352;      // 32: T_hi R_hi + T_lo R_hi | T_hi R_lo
    static constexpr uint32_t tm_o2 = 384;     // [2] x 32
    static constexpr uint32_t tm_u = 448;      // [2] x 32: U hi | lo
    static constexpr uint32_t tmem_cols = 512;
    static_assert(stage_bytes % 1024 == 0 && s_off % 1024 == 0 && s_half_bytes % 1024 == 0 && v_off % 1024 == 0, "swizzled regions: 1024-byte alignment");
    static_assert(a_off % 1024 == 0 && 2 * a_term_bytes >= q_bytes, "the K tile of an owned chunk lands in the staging matrix");
    static_assert(total <= 232448, "shared memory budget");
};

struct GdnBars {
    int full, empty, v_full, v_read, s_full, g_done, kg_full, t_free, t_ack, t_staged, p_done, a_full, x_done, x_read, y_done, y_free, t_full, r_full, w_done,
        w_read, wv_full, wt_full, o2_done, o2_free, u_done, u_empty, g_full, g_empty, row_ready, count;
};
template <int DK>
__device__ __forceinline__ constexpr GdnBars gdn_bars() {
    using L = GdnCfg<DK>;
    GdnBars b{};
    int i = 0;
    b.full = i; i += L::NS;
    b.empty = i; i += L::NS;
    b.v_full = i; i += L::NV;
    b.v_read = i; i += L::NV;
    b.s_full = i; i += 2;
    b.g_done = i; i += 1;
    b.kg_full = i; i += 1;
    b.t_free = i; i += 2;
    b.t_ack = i; i += 1;
    b.t_staged = i; i += 1;
    b.p_done = i; i += 2;
    b.a_full = i; i += 2;
    b.x_done = i; i += 1;
    b.x_read = i; i += 1;
    b.y_done = i; i += 2;
    b.y_free = i; i += 2;
    b.t_full = i; i += 2;
    b.r_full = i; i += 1;
    b.w_done = i; i += 2;
    b.w_read = i; i += 1;
    b.wv_full = i; i += 2;
    b.wt_full = i; i += 1;
    b.o2_done = i; i += 2;
    b.o2_free = i; i += 2;
    b.u_done = i; i += 2;
    b.u_empty = i; i += 2;
    b.g_full = i; i += 2;
    b.g_empty = i; i += 2;
    b.row_ready = i; i += 4;
    b.count = i;
    return b;
}

template <int DK>
__global__ void __launch_bounds__(GdnCfg<DK>::kThreads, 1)
esc_gdn_scan_kernel(const __grid_constant__ CUtensorMap tq, const __grid_constant__ CUtensorMap tk, const __grid_constant__ CUtensorMap tv,
                    const float* __restrict__ g, const float* __restrict__ beta, const float* state_in, float* state_out,
                    float* __restrict__ o, uint32_t H, uint32_t DV, uint64_t T, uint64_t t_stride) {
    using L = GdnCfg<DK>;
    constexpr GdnBars BI = gdn_bars<DK>();
    static_assert(BI.count <= 64, "barrier area");
    constexpr int NS = L::NS, NV = L::NV, W = kGW;

    extern __shared__ uint8_t smem_raw[];
    uint8_t* sm = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sm_a = smem_u32(sm);
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + L::bar_off);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sm + L::bar_off + 64 * 8);
    float* gate = reinterpret_cast<float*>(sm + L::gate_off);   // [2][3][256]: b2, eb, beta per slot

    // (the shuffle tells the compiler that the warp index is warp-uniform: the role branches become uniform branches, and
    // inside them descriptors and addresses can live in uniform registers instead of being moved there before every MMA)
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    const uint32_t bh = blockIdx.y, b = bh / H, h = bh % H, dv0 = blockIdx.x * W;
    const uint32_t n_chunks = (uint32_t)((T + kGC - 1) / kGC);
    const int q = warp & 3;   // TMEM lane quadrant this warp may access
    const int g8 = lane >> 2, t4 = lane & 3;
    // the d_v slices of one (b, h) form a thread-block cluster: T = (I + A^k)^-1 depends on k, beta and the decays only, so CTA
    // c % csz computes the T of chunk c ("owns" it) and pushes it into every CTA's operand ring
    const uint32_t csz = cluster_nctarank(), rank = cluster_ctarank();

    // Programmatic dependent launch: the next kernel of the stream (typically the next layer's scan) may start its on-chip setup
    // while this one runs; everything this kernel reads from or writes to global memory comes after griddepcontrol.wait below.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // ---- one-time setup ------------------------------------------------------------------------------------
    if (warp == 0 && lane == 0) {
        for (int i = 0; i < NS; ++i) { mbar_init(&bars[BI.full + i], 1); mbar_init(&bars[BI.empty + i], 2); }
        for (int i = 0; i < NV; ++i) { mbar_init(&bars[BI.v_full + i], 1); mbar_init(&bars[BI.v_read + i], 4); }
        mbar_init(&bars[BI.x_done], 1); mbar_init(&bars[BI.x_read], 4);
        mbar_init(&bars[BI.r_full], 4); mbar_init(&bars[BI.w_read], 4); mbar_init(&bars[BI.wt_full], 4);
        for (int i = 0; i < 4; ++i) mbar_init(&bars[BI.row_ready + i], 1);
        mbar_init(&bars[BI.g_done], 1); mbar_init(&bars[BI.kg_full], 1); mbar_init(&bars[BI.t_ack], csz); mbar_init(&bars[BI.t_staged], 1);
        for (int i = 0; i < 2; ++i) {
            mbar_init(&bars[BI.s_full + i], 4);
            mbar_init(&bars[BI.t_free + i], csz);
            mbar_init(&bars[BI.p_done + i], 1); mbar_init(&bars[BI.a_full + i], 4);
            mbar_init(&bars[BI.y_done + i], 1); mbar_init(&bars[BI.y_free + i], 4);
            mbar_init(&bars[BI.t_full + i], 1);
            mbar_init(&bars[BI.w_done + i], 1);
            mbar_init(&bars[BI.wv_full + i], 4);
            mbar_init(&bars[BI.o2_done + i], 1); mbar_init(&bars[BI.o2_free + i], 4);
            mbar_init(&bars[BI.u_done + i], 1); mbar_init(&bars[BI.u_empty + i], 4);
            mbar_init(&bars[BI.g_full + i], 1); mbar_init(&bars[BI.g_empty + i], 16);
        }
        fence_mbar_init();
        tma_prefetch_desc(&tq); tma_prefetch_desc(&tk); tma_prefetch_desc(&tv);
    }
    if (warp == 2) tmem_alloc(tmem_slot, L::tmem_cols);
    // Without a cluster (csz = 1: calls of up to kGdnShortT tokens, ONE chunk) there is nobody to push to: the T warps write the
    // inverse straight into operand slot 0 and arrive on its barrier themselves (no staging, no push, no slot flow control).
    const bool direct = csz == 1;
    if (direct && n_chunks > 1) __trap();   // the host launches without a cluster for one-chunk calls only
    // the T staging buffer (the slot in direct mode): the blocks above the diagonal are never written, so they are zeroed once
    for (uint32_t i = threadIdx.x; i < L::t_bytes / 16; i += L::kThreads)
        reinterpret_cast<uint4*>(sm + (direct ? L::t_off : L::tstage_off))[i] = make_uint4(0, 0, 0, 0);
    fence_proxy_async_smem();
    tc_fence_before_sync();
    cluster_sync();   // every CTA's barriers are initialised before a peer copies a T into it or arrives on them
    tc_fence_after_sync();
    asm volatile("griddepcontrol.wait;" ::: "memory");   // ---- global memory may be touched from here on ----
    const uint32_t tb = __shfl_sync(0xffffffffu, *tmem_slot, 0);
    GPROF_DECL

    if (warp == 0) {
        // ================= TMA producer =================
        if (lane == 0) {
            auto prefetch_chunk = [&](uint32_t c) {
                const int t0 = (int)(c * kGC);
                tma_prefetch_5d(&tq, 0, t0, 0, (int)h, (int)b);
                tma_prefetch_5d(&tk, 0, t0, 0, (int)h, (int)b);
                tma_prefetch_4d(&tv, (int)dv0, (int)h, t0, (int)b);
            };
            for (uint32_t c = NS; c < n_chunks && c < (uint32_t)(NS + kGAhead); ++c) prefetch_chunk(c);
            for (uint32_t c = 0; c < n_chunks; ++c) {
                if (c + NS + kGAhead < n_chunks) prefetch_chunk(c + NS + kGAhead);
                const uint32_t s = c % NS, vi = c % NV;
                const int t0 = (int)(c * kGC);
                uint8_t* st = sm + L::stage_off + s * L::stage_bytes;
                if (c >= (uint32_t)NS) GW_(0, mbar_wait_relaxed(&bars[BI.empty + s], ((c / NS) & 1) ^ 1));
                uint64_t* full = &bars[BI.full + s];
                mbar_arrive_expect_tx(full, 2 * L::q_bytes);
                tma_load_5d(st, &tq, full, 0, t0, 0, (int)h, (int)b);
                tma_load_5d(st + L::q_bytes, &tk, full, 0, t0, 0, (int)h, (int)b);
                if (c >= (uint32_t)NV) GW_(1, mbar_wait_relaxed(&bars[BI.v_read + vi], ((c / NV) & 1) ^ 1));
                mbar_arrive_expect_tx(&bars[BI.v_full + vi], L::v_bytes);
                tma_load_4d(sm + L::v_off + vi * L::v_bytes, &tv, &bars[BI.v_full + vi], (int)dv0, (int)h, t0, (int)b);
            }
            // tail: the last commits have reached this CTA's stage barriers before anyone may exit
            for (uint32_t c = n_chunks > (uint32_t)NS ? n_chunks - NS : 0; c < n_chunks; ++c) mbar_wait(&bars[BI.empty + c % NS], (c / NS) & 1);
        }
    } else if (warp == 1) {
        // ================= gate warp: b2_i = sum_{r<=i in chunk} log2 a_r, eb = 2^b2, beta; 256 tokens per batch =================
        // (the per-token loops are rolled through shared memory on purpose: this warp runs once per four chunks and its code
        // must not evict the per-chunk loops of the other roles from the instruction cache)
        const uint32_t n_batches = (uint32_t)((T + kGBatch - 1) / kGBatch);
        constexpr int GL = kGC / 8;   // lanes per chunk
        float* raw = reinterpret_cast<float*>(sm + L::raw_off);   // [2][a[256], beta[256]]: asynchronous copies, one batch ahead
        auto load_g = [&](uint32_t bt) {
            float* ra_ = raw + (bt & 1) * 2 * kGBatch;
#pragma unroll 1
            for (int u = 0; u < 8; ++u) {
                const uint64_t tt = (uint64_t)bt * kGBatch + lane + 32 * u;
                if (tt < T) {
                    const size_t idx = ((size_t)b * t_stride + tt) * H + h;
                    cp_async_4(ra_ + lane + 32 * u, g + idx);
                    cp_async_4(ra_ + kGBatch + lane + 32 * u, beta + idx);
                } else {   // tokens beyond T: a = 1, beta = 0 (k = q = v = 0 by the TMA fill): identity
                    ra_[lane + 32 * u] = 1.f;
                    ra_[kGBatch + lane + 32 * u] = 0.f;
                }
            }
            cp_async_commit();
        };
        if (n_batches) load_g(0);
        for (uint32_t bt = 0; bt < n_batches; ++bt) {
            const uint32_t slot = bt & 1;
            cp_async_wait_all();
            __syncwarp();
            if (bt >= 2) GW_(0, mbar_wait_relaxed(&bars[BI.g_empty + slot], ((bt >> 1) & 1) ^ 1));
            float* b2 = gate + slot * 3 * kGBatch;
            float* eb = b2 + kGBatch;
            float* be = eb + kGBatch;
            const float* ra_ = raw + slot * 2 * kGBatch;
            float run = 0.f;   // lane owns tokens 8 lane .. 8 lane + 7: local inclusive sums, then a segmented scan over the 8 lanes of a chunk
#pragma unroll 1
            for (int u = 0; u < 8; ++u) {
                run += log2f(ra_[8 * lane + u]);
                b2[8 * lane + u] = run;
                be[8 * lane + u] = ra_[kGBatch + 8 * lane + u];
            }
            __syncwarp();
            if (bt + 1 < n_batches) load_g(bt + 1);   // next batch's copies fly while the consumers work on this one
            float incl = run;
#pragma unroll
            for (int d = 1; d < GL; d <<= 1) {
                const float up = __shfl_up_sync(0xffffffffu, incl, d);
                if ((lane % GL) >= d) incl += up;
            }
            const float prev = __shfl_up_sync(0xffffffffu, incl, 1);
            const float excl = (lane % GL) ? prev : 0.f;
#pragma unroll 1
            for (int u = 0; u < 8; ++u) {
                const float x = excl + b2[8 * lane + u];
                b2[8 * lane + u] = x;
                eb[8 * lane + u] = ex2(x);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BI.g_full + slot]);
        }
    } else if (warp == 2) {
        // ================= issuer: P = Q K^T  (G = K K^T is issued by the T warps, for the chunks this CTA inverts) =================
        constexpr uint32_t idPG = idesc_bf16(kGC, kGC, 0, 0);
        const uint64_t dQ0 = smem_desc(sm_a + L::stage_off, 16, 1024, kSwz128);
        const uint64_t dK0 = smem_desc(sm_a + L::stage_off + L::q_bytes, 16, 1024, kSwz128);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t s = c % NS, pb = c & 1;
            GW_(0, mbar_wait_relaxed(&bars[BI.full + s], (c / NS) & 1));
            const uint64_t dQ = smem_desc_advance(dQ0, s * L::stage_bytes), dK = smem_desc_advance(dK0, s * L::stage_bytes);
            if (c >= 2) GW_(2, mbar_wait_relaxed(&bars[BI.o2_done + pb], ((c - 2) >> 1) & 1));           // O2(c - 2) has read A^q from buffer pb
            tc_fence_after_sync();
#pragma unroll 1
            for (int ks = 0; ks < DK / 16; ++ks) {
                const uint32_t adv = (ks / 4) * L::half_bytes + (ks % 4) * 32;
                mma_bf16_ss_w(tb + L::tm_p + pb * kGC, smem_desc_advance(dQ, adv), smem_desc_advance(dK, adv), idPG, ks > 0);
            }
            mma_commit_w(&bars[BI.p_done + pb]);
            mma_commit_w(&bars[BI.empty + s]);
        }
    } else if (warp == 3) {
        // ================= issuer of the chain: [X|.] = K [S_hi|S_lo], [Y|.] = Q [S_hi|S_lo], Wm = T R, U = K^T W~ =================
        constexpr uint32_t idXY = idesc_bf16(kGC, 2 * W, 0, 0);
        constexpr uint32_t idW2 = idesc_bf16(kGC, 2 * W, 1, 1);   // T_hi [R_hi | R_lo]
        constexpr uint32_t idW1 = idesc_bf16(kGC, W, 1, 1);       // T_lo R_hi
        constexpr uint32_t idU = idesc_bf16(DK, 2 * W, 1, 1);
        const uint64_t dQ0 = smem_desc(sm_a + L::stage_off, 16, 1024, kSwz128);
        const uint64_t dK0 = smem_desc(sm_a + L::stage_off + L::q_bytes, 16, 1024, kSwz128);
        const uint64_t dKt0 = smem_desc(sm_a + L::stage_off + L::q_bytes, L::half_bytes, 1024, kSwz128);   // K^T: MN-major
        const uint64_t dS0 = smem_desc(sm_a + L::s_off, 16, 1024, kSwz128);
        const uint64_t dT0 = smem_desc(sm_a + L::t_off, 128, L::op_sbo, kSwzNone);
        const uint64_t dR = smem_desc(sm_a + L::r_off, 128, L::op_sbo, kSwzNone);
        const uint64_t dWt = smem_desc(sm_a + L::wt_off, 128, L::op_sbo, kSwzNone);
        constexpr uint32_t idO2 = idesc_bf16(kGC, 2 * W, 0, 1);
        constexpr uint32_t idO1 = idesc_bf16(kGC, W, 0, 1);
        const uint64_t dW0 = smem_desc(sm_a + L::wv_off, 128, L::op_sbo, kSwzNone);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t s = c % NS, sb = c & 1;
            if (lane == 0 && !direct) mbar_arrive_expect_tx(&bars[BI.t_full + sb], L::t_bytes);   // T(c): pushed by CTA c % csz (bulk copy into slot sb)
            GW_(0, mbar_wait(&bars[BI.full + s], (c / NS) & 1));
            if (c >= 1) GW_(1, mbar_wait(&bars[BI.x_read], (c - 1) & 1));
            GW_(2, mbar_wait(&bars[BI.s_full + sb], (c >> 1) & 1));
            tc_fence_after_sync();
            const uint64_t dQ = smem_desc_advance(dQ0, s * L::stage_bytes), dK = smem_desc_advance(dK0, s * L::stage_bytes);
            const uint64_t dS = smem_desc_advance(dS0, sb * L::s_bytes);
#pragma unroll
            for (int ks = 0; ks < DK / 16; ++ks)
                mma_bf16_ss_w(tb + L::tm_x, smem_desc_advance(dK, (ks / 4) * L::half_bytes + (ks % 4) * 32),
                              smem_desc_advance(dS, (ks / 4) * L::s_half_bytes + (ks % 4) * 32), idXY, ks > 0);
            mma_commit_w(&bars[BI.x_done]);
            if (c >= 2) GW_(3, mbar_wait(&bars[BI.y_free + sb], ((c - 2) >> 1) & 1));
            tc_fence_after_sync();
#pragma unroll
            for (int ks = 0; ks < DK / 16; ++ks)
                mma_bf16_ss_w(tb + L::tm_y + sb * 2 * W, smem_desc_advance(dQ, (ks / 4) * L::half_bytes + (ks % 4) * 32),
                              smem_desc_advance(dS, (ks / 4) * L::s_half_bytes + (ks % 4) * 32), idXY, ks > 0);
            mma_commit_w(&bars[BI.y_done + sb]);
            // Wm = T R
            GW_(4, mbar_wait(&bars[BI.t_full + sb], (c >> 1) & 1));
            if (c >= 1) GW_(1, mbar_wait(&bars[BI.w_read], (c - 1) & 1));
            GW_(5, mbar_wait(&bars[BI.r_full], c & 1));
            tc_fence_after_sync();
            const uint64_t dT = smem_desc_advance(dT0, sb * L::t_bytes);
#pragma unroll
            for (int ks = 0; ks < kGC / 16; ++ks)
                mma_bf16_ss_w(tb + L::tm_w, smem_desc_advance(dT, 2 * ks * 128), smem_desc_advance(dR, 2 * ks * 128), idW2, ks > 0);
#pragma unroll
            for (int ks = 0; ks < kGC / 16; ++ks)
                mma_bf16_ss_w(tb + L::tm_w, smem_desc_advance(dT, L::t_term_bytes + 2 * ks * 128), smem_desc_advance(dR, 2 * ks * 128), idW1, 1);
            mma_commit_w(&bars[BI.w_done + sb]);
            // U = K^T W~
            if (c >= 2) GW_(6, mbar_wait(&bars[BI.u_empty + sb], ((c - 2) >> 1) & 1));
            GW_(6, mbar_wait(&bars[BI.wt_full], c & 1));
            tc_fence_after_sync();
            const uint64_t dKt = smem_desc_advance(dKt0, s * L::stage_bytes);
#pragma unroll
            for (int ks = 0; ks < kGC / 16; ++ks)
                mma_bf16_ss_w(tb + L::tm_u + sb * 2 * W, smem_desc_advance(dKt, 2 * ks * 1024), smem_desc_advance(dWt, 2 * ks * 128), idU, ks > 0);
            mma_commit_w(&bars[BI.u_done + sb]);
            mma_commit_w(&bars[BI.empty + s]);
            // O2 = A^q_hi [Wm_hi | Wm_lo] + A^q_lo Wm_hi (A operand from TMEM).  Issued from this warp in the gap before S(c + 1) is
            // ready: its operands (A^q(c) from the score warps, the Wm operand written together with W~) are there by now.
            if (c >= 2) GW_(3, mbar_wait(&bars[BI.o2_free + sb], ((c - 2) >> 1) & 1));
            GW_(3, mbar_wait(&bars[BI.a_full + sb], (c >> 1) & 1));
            GW_(3, mbar_wait(&bars[BI.wv_full + sb], (c >> 1) & 1));
            tc_fence_after_sync();
            {
                const uint64_t dWv = smem_desc_advance(dW0, sb * L::op_bytes);
                const uint32_t dO = tb + L::tm_o2 + sb * 2 * W, aA = tb + L::tm_p + sb * kGC;
#pragma unroll
                for (int ks = 0; ks < kGC / 16; ++ks) mma_bf16_ts_w(dO, aA + 16 * ks, smem_desc_advance(dWv, 2 * ks * 128), idO2, ks > 0);
#pragma unroll
                for (int ks = 0; ks < kGC / 16; ++ks) mma_bf16_ts_w(dO, aA + 16 * ks + 8, smem_desc_advance(dWv, 2 * ks * 128), idO1, 1);
                mma_commit_w(&bars[BI.o2_done + sb]);
            }
        }
    } else if (warp == 4) {
        // ================= ack warp: tells the owners of T(c + 2) and T(c) that this CTA's Wm(c) has read its copy of T(c) =================
        // (a remote arrive costs its thread ~1000 cycles: on a warp of its own it is off every other role's path)
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t sb = c & 1;
            GW_(0, mbar_wait_relaxed(&bars[BI.w_done + sb], (c >> 1) & 1));
            if (lane == 0) {
                if (c + 2 < n_chunks) mbar_arrive_cluster_relaxed(mapa(smem_u32(&bars[BI.t_free + sb]), (c + 2) % csz));   // slot sb is free for T(c + 2)
                mbar_arrive_cluster_relaxed(mapa(smem_u32(&bars[BI.t_ack]), c % csz));                                       // the owner's staging copy has landed
            }
            __syncwarp();
        }
    } else if (warp == 5) {
        // ================= push warp: T(c) of an owned chunk, staged by the T warps -> slot c % 2 of every CTA of the cluster =================
        // Slot c % 2 of every CTA is free once every CTA's Wm(c - 2) has completed.  Arrivals on this CTA's t_free come for the chunks it
        // owns only (all of the same parity when csz is even; without a cluster, csz = 1, every chunk), one phase per owned chunk c >= 2.  (On a warp of its own: the T warps
        // are typically a few chunks ahead of the chain, and waiting for the slot would hold up their next chunk.)
        uint32_t k_own = 0;
        for (uint32_t c = rank; c < n_chunks && !direct; c += csz, ++k_own) {
            GW_(0, mbar_wait_relaxed(&bars[BI.t_staged], k_own & 1));
            // phase of t_free[c % 2] here: the owned chunks before this one that used the slot and had a predecessor (c' >= 2)
            if (c >= 2) GW_(1, mbar_wait_relaxed(&bars[BI.t_free + (c & 1)], (csz > 1 ? k_own - (rank < 2 ? 1u : 0u) : (c - 2) >> 1) & 1));
            if (lane == 0) {
                const uint32_t dst = sm_a + L::t_off + (c & 1) * L::t_bytes, full = smem_u32(&bars[BI.t_full + (c & 1)]);
                for (uint32_t pr = 0; pr < csz; ++pr) bulk_copy_to_cluster(mapa(dst, pr), sm_a + L::tstage_off, L::t_bytes, mapa(full, pr));
            }
            __syncwarp();
        }
    } else if (warp >= 8 && warp < 12) {
        // ================= T warps: A^k = beta_i D_ij G_ij (j < i), T = (I + A^k)^-1 -> MN-major A operand =================
        // T depends on k, beta and the decays only: the same matrix in every d_v slice of a head.  The slices of a head are a
        // cluster; CTA c % csz computes T(c) — these four warps, one chunk in csz, far ahead of the carry chain — into a staging
        // buffer and pushes it into operand slot c % 2 of EVERY CTA of the cluster (bulk copies over distributed shared memory,
        // completion as transaction bytes on each CTA's t_full barrier).  (The first r02 version computed every T in every CTA:
        // two sets of four warps, and the chain still waited ~800 cycles per chunk for them.)  The pipeline of an owned chunk is
        // self-contained: own gate values (the gate warp's ring only runs a few chunks ahead of the chain), own TMA load of the K
        // tile (into the staging matrix, which is free until A^k is formed), G = K K^T issued by warp 8.
        // One 64 x 64 bf16 staging matrix (hi and lo terms, row-major, padded rows) holds the blocks of A^k below the diagonal
        // and the blocks of U = T^T on and above it: warp I writes block row I of both and reads the A^k blocks and the
        // diagonal blocks of the rows below it, row by row as they become ready (one mbarrier per row).  The loops over blocks are
        // rolled on purpose (the first version unrolled them: 84 KB of SASS per kernel, every role starved by instruction-cache
        // misses, r02 ncu: 5.5 warps stalled on "no instruction" per issue).
        const int I = q;                                   // block row of A^k this warp forms = block row of U it fills
        const int ia = 16 * I + g8, ib = ia + 8;
        float* lt = reinterpret_cast<float*>(sm + L::lt_off) + I * 16 * L::lt_pitch;   // fp32 diagonal block, transposed: lt[j][i]
        float* b2 = reinterpret_cast<float*>(sm + L::tg_off) + I * 2 * kGC;           // this warp's copy of the chunk's gate values
        float* be = b2 + kGC;
        const uint32_t mi = lane >> 3, rr = lane & 7;
        // ldmatrix row addresses inside a 16 x 16 block, by the order of the four 8 x 8 matrices:
        //   "rc": (rows 0-7, cols 0-7), (rows 8-15, cols 0-7), (rows 0-7, cols 8-15), (rows 8-15, cols 8-15)
        //   "cr": (rows 0-7, cols 0-7), (rows 0-7, cols 8-15), (rows 8-15, cols 0-7), (rows 8-15, cols 8-15)
        const uint32_t rc_lane = (rr + 8 * (mi & 1)) * L::a_pitch + 16 * (mi >> 1);
        const uint32_t cr_lane = (rr + 8 * (mi >> 1)) * L::a_pitch + 16 * (mi & 1);
        auto blk = [](int r, int cc) { return (uint32_t)((16 * r) * L::a_pitch + (16 * cc) * 2); };
        uint8_t* ast = sm + L::a_off;
        const uint32_t a_hi = sm_a + L::a_off, a_lo = a_hi + L::a_term_bytes;
        uint8_t* tbase = sm + (direct ? L::t_off : L::tstage_off);
        constexpr uint32_t idG = idesc_bf16(kGC, kGC, 0, 0);
        const uint64_t dKg = smem_desc(sm_a + L::a_off, 16, 1024, kSwz128);
        uint32_t k_own = 0;                                // owned chunks done: the phase of this pipeline's own barriers
        // raw a / beta of owned chunk number k (chunk cc) -> traw[k & 1], by warp 8: asynchronous copies, waited for before the
        // barrier that ends the preceding owned chunk.  Tokens beyond T: a = 1, beta = 0 (identity).
        auto load_raw = [&](uint32_t cc, uint32_t k) {
            float* raw = reinterpret_cast<float*>(sm + L::traw_off) + (k & 1) * 2 * kGC;
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const uint64_t tt = (uint64_t)cc * kGC + lane + 32 * u;
                if (tt < T) {
                    const size_t idx = ((size_t)b * t_stride + tt) * H + h;
                    cp_async_4(raw + lane + 32 * u, g + idx);
                    cp_async_4(raw + kGC + lane + 32 * u, beta + idx);
                } else {
                    raw[lane + 32 * u] = 1.f;
                    raw[kGC + lane + 32 * u] = 0.f;
                }
            }
            cp_async_commit();
        };
        // the K tile of an owned chunk -> the staging matrix (free from the barrier that ends the preceding owned chunk until A^k is
        // formed); issued right after that barrier, so that the load flies during the push and the gate values
        auto load_k = [&](uint32_t cc) {
            mbar_arrive_expect_tx(&bars[BI.kg_full], L::q_bytes);
            tma_load_5d(sm + L::a_off, &tk, &bars[BI.kg_full], 0, (int)(cc * kGC), 0, (int)h, (int)b);
        };
        if (rank < n_chunks) {
            if (I == 0) {
                if (lane == 0) load_k(rank);
                load_raw(rank, 0);
                cp_async_wait_all();
            }
            named_bar_sync(1, 128);
        }
        for (uint32_t c = rank; c < n_chunks; c += csz, ++k_own) {
            GSEG_START
            if (I == 0 && c + csz < n_chunks) load_raw(c + csz, k_own + 1);
            if (I == 0) {   // G = K K^T, issued first: the MMAs run while the gate values are formed
                mbar_wait(&bars[BI.kg_full], k_own & 1);
                tc_fence_after_sync();
#pragma unroll 1
                for (int ks = 0; ks < DK / 16; ++ks) {
                    const uint32_t adv = (ks / 4) * L::half_bytes + (ks % 4) * 32;
                    mma_bf16_ss_w(tb + L::tm_g, smem_desc_advance(dKg, adv), smem_desc_advance(dKg, adv), idG, ks > 0);
                }
                mma_commit_w(&bars[BI.g_done]);
            }
            // gate values of the chunk from the raw a / beta that warp 8 copied in one owned chunk ahead (cp.async): lane l owns
            // tokens 2 l, 2 l + 1, then a warp scan.  (Each of the four warps keeps its own copy: no barrier.  The summation order
            // differs from the gate warp's, so these b agree with the chain's to an ulp of the exponent, not bit for bit; both are
            // functions of the chunk's inputs only.)
            {
                const float* raw = reinterpret_cast<const float*>(sm + L::traw_off) + (k_own & 1) * 2 * kGC;
                const float2 gv = *reinterpret_cast<const float2*>(raw + 2 * lane);
                const float2 bv = *reinterpret_cast<const float2*>(raw + kGC + 2 * lane);
                const float l0 = log2f(gv.x), l1 = l0 + log2f(gv.y);
                float incl = l1;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const float up = __shfl_up_sync(0xffffffffu, incl, d);
                    if (lane >= d) incl += up;
                }
                const float excl = incl - l1;
                *reinterpret_cast<float2*>(b2 + 2 * lane) = make_float2(excl + l0, excl + l1);
                *reinterpret_cast<float2*>(be + 2 * lane) = bv;
                __syncwarp();
            }
            const float bia = b2[ia], bib = b2[ib], bea = be[ia], beb = be[ib];
            GSEG(0);
            mbar_wait(&bars[BI.g_done], k_own & 1);   // (the MMAs have also finished reading the K tile: the staging matrix is free)
            tc_fence_after_sync();
            GSEG(1);
            uint32_t cur[8], nxt[8];
            tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_g + 16 * I), cur);
            if (I > 0) tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_g), nxt);
            tmem_ld_wait();
            // the diagonal block in fp32, transposed and masked (j < i), for the substitution
#pragma unroll
            for (int jb = 0; jb < 2; ++jb) {
                const int jl = 8 * jb + 2 * t4, j0 = 16 * I + jl;
                const float2 bj = *reinterpret_cast<const float2*>(b2 + j0);
                float a0 = bea * ex2(bia - bj.x) * __uint_as_float(cur[4 * jb + 0]);
                float a1 = bea * ex2(bia - bj.y) * __uint_as_float(cur[4 * jb + 1]);
                float c0 = beb * ex2(bib - bj.x) * __uint_as_float(cur[4 * jb + 2]);
                float c1 = beb * ex2(bib - bj.y) * __uint_as_float(cur[4 * jb + 3]);
                a0 = (j0 < ia) ? a0 : 0.f;
                a1 = (j0 + 1 < ia) ? a1 : 0.f;
                c0 = (j0 < ib) ? c0 : 0.f;
                c1 = (j0 + 1 < ib) ? c1 : 0.f;
                lt[jl * L::lt_pitch + g8] = a0;
                lt[(jl + 1) * L::lt_pitch + g8] = a1;
                lt[jl * L::lt_pitch + g8 + 8] = c0;
                lt[(jl + 1) * L::lt_pitch + g8 + 8] = c1;
            }
            // rows ia, ib of A^k left of the diagonal, 16 columns at a time (the next block's TMEM load flies meanwhile)
#pragma unroll 1
            for (int m2 = 0; m2 < I; ++m2) {
#pragma unroll
                for (int i = 0; i < 8; ++i) cur[i] = nxt[i];
                if (m2 + 1 < I) tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_g + 16 * (m2 + 1)), nxt);
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {
                    const int j0 = 16 * m2 + 8 * jb + 2 * t4;
                    const float2 bj = *reinterpret_cast<const float2*>(b2 + j0);
                    const float a0 = bea * ex2(bia - bj.x) * __uint_as_float(cur[4 * jb + 0]);
                    const float a1 = bea * ex2(bia - bj.y) * __uint_as_float(cur[4 * jb + 1]);
                    const float c0 = beb * ex2(bib - bj.x) * __uint_as_float(cur[4 * jb + 2]);
                    const float c1 = beb * ex2(bib - bj.y) * __uint_as_float(cur[4 * jb + 3]);
                    uint32_t lo0, lo1;
                    const uint32_t hi0 = split2(a0, a1, lo0), hi1 = split2(c0, c1, lo1);
                    const uint32_t oa = ia * L::a_pitch + j0 * 2, ob = ib * L::a_pitch + j0 * 2;
                    *reinterpret_cast<uint32_t*>(ast + oa) = hi0;
                    *reinterpret_cast<uint32_t*>(ast + L::a_term_bytes + oa) = lo0;
                    *reinterpret_cast<uint32_t*>(ast + ob) = hi1;
                    *reinterpret_cast<uint32_t*>(ast + L::a_term_bytes + ob) = lo1;
                }
                tmem_ld_wait();
            }
            tc_fence_before_sync();
            GSEG(3);
            // T_II = (I + A_II)^-1, column by column: lane col solves (I + A_II) x = e_col by forward substitution in fp32
            // (right-looking: once x_j is final every later row takes its term; independent FMAs, the dependency chain is one FMA
            // per step; the columns of A_II are warp-wide broadcast reads).  Unrolled on purpose: the rolled form with one row per
            // lane (a shuffle and an FMA per step on the chain) took 180 cycles per step, 40 % of this warp's time (r02 ncu).
            {
                const int col = lane & 15;
                float x[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) x[i] = (i == col) ? 1.f : 0.f;
#pragma unroll
                for (int j = 0; j + 1 < 16; ++j) {
#pragma unroll
                    for (int i4 = (j + 1) / 4; i4 < 4; ++i4) {
                        const float4 l4 = *reinterpret_cast<const float4*>(&lt[j * L::lt_pitch + 4 * i4]);
                        if (4 * i4 + 0 > j) x[4 * i4 + 0] = fmaf(-l4.x, x[j], x[4 * i4 + 0]);
                        if (4 * i4 + 1 > j) x[4 * i4 + 1] = fmaf(-l4.y, x[j], x[4 * i4 + 1]);
                        if (4 * i4 + 2 > j) x[4 * i4 + 2] = fmaf(-l4.z, x[j], x[4 * i4 + 2]);
                        if (4 * i4 + 3 > j) x[4 * i4 + 3] = fmaf(-l4.w, x[j], x[4 * i4 + 3]);
                    }
                }
                // lane col holds column col of T_II = row col of U_II = T_II^T: 16 consecutive rows i of T
                uint32_t hi[8], lo[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) hi[e] = split2(x[2 * e], x[2 * e + 1], lo[e]);
                // the T staging buffer still holds T(c - csz): it may be rewritten once every CTA's copy of it has landed (t_ack: every
                // CTA's Wm(c - csz) has completed).  Waited for here, at the first write, not at the top: the push, the peers' Wm and
                // their acknowledgement take ~4000 cycles, which the gate values, the K tile, G, A^k and the substitution overlap.
                if (k_own >= 1) mbar_wait_relaxed(&bars[BI.t_ack], (k_own - 1) & 1);
                if (lane < 16) {
                    uint8_t* dh = ast + blk(I, I) + col * L::a_pitch;   // U_II row-major in the staging matrix
                    *reinterpret_cast<uint4*>(dh) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                    *reinterpret_cast<uint4*>(dh + 16) = make_uint4(hi[4], hi[5], hi[6], hi[7]);
                    *reinterpret_cast<uint4*>(dh + L::a_term_bytes) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
                    *reinterpret_cast<uint4*>(dh + L::a_term_bytes + 16) = make_uint4(lo[4], lo[5], lo[6], lo[7]);
                    // T[i][j], j = 16 I + col, i = 16 I + 0..15 -> (i/8) op_sbo + (j/8) 128 + (j%8) 16 + (i%8) 2
                    const uint32_t j = 16 * I + col;
                    uint8_t* th = tbase + (2 * I) * L::op_sbo + (j >> 3) * 128 + (j & 7) * 16;
                    *reinterpret_cast<uint4*>(th) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                    *reinterpret_cast<uint4*>(th + L::op_sbo) = make_uint4(hi[4], hi[5], hi[6], hi[7]);
                    *reinterpret_cast<uint4*>(th + L::t_term_bytes) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
                    *reinterpret_cast<uint4*>(th + L::t_term_bytes + L::op_sbo) = make_uint4(lo[4], lo[5], lo[6], lo[7]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BI.row_ready + I]);   // block row I of A^k and U_II are staged
            GSEG(4);
            // block row I of U = T^T:  U_I,Ic = -(sum_{K=I}^{Ic-1} U_I,K (A^k_{Ic,K})^T) U_Ic,Ic.  (The three hi / lo terms of a
            // product accumulate in place: separate accumulators shorten the mma chain but cost more instructions than they save.)
#pragma unroll 1
            for (int Ic = I + 1; Ic < 4; ++Ic) {
                mbar_wait(&bars[BI.row_ready + Ic], k_own & 1);
                float z[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll 1
                for (int K = I; K < Ic; ++K) {
                    uint32_t xh[4], xl[4], bhh[4], bll[4];
                    ldmatrix_x4(xh, a_hi + blk(I, K) + rc_lane);
                    ldmatrix_x4(xl, a_lo + blk(I, K) + rc_lane);
                    ldmatrix_x4(bhh, a_hi + blk(Ic, K) + cr_lane);
                    ldmatrix_x4(bll, a_lo + blk(Ic, K) + cr_lane);
#pragma unroll
                    for (int nt = 0; nt < 2; ++nt) {
                        mma_sync_16816(z[nt], xl, bhh[2 * nt], bhh[2 * nt + 1]);
                        mma_sync_16816(z[nt], xh, bll[2 * nt], bll[2 * nt + 1]);
                        mma_sync_16816(z[nt], xh, bhh[2 * nt], bhh[2 * nt + 1]);
                    }
                }
                uint32_t zh[4], zl[4], uh[4], ul[4];
#pragma unroll
                for (int nt = 0; nt < 2; ++nt)
#pragma unroll
                    for (int hf = 0; hf < 2; ++hf)
                        zh[2 * nt + hf] = split2(z[nt][2 * hf], z[nt][2 * hf + 1], zl[2 * nt + hf]);
                ldmatrix_x4_trans(uh, a_hi + blk(Ic, Ic) + rc_lane);   // B fragments of U_Ic,Ic (row-major [k][n]: transposing load)
                ldmatrix_x4_trans(ul, a_lo + blk(Ic, Ic) + rc_lane);
                float y[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) {
                    mma_sync_16816(y[nt], zl, uh[2 * nt], uh[2 * nt + 1]);
                    mma_sync_16816(y[nt], zh, ul[2 * nt], ul[2 * nt + 1]);
                    mma_sync_16816(y[nt], zh, uh[2 * nt], uh[2 * nt + 1]);
                }
                // U_I,Ic = -y: rows r = g8 / g8 + 8 (j = 16 I + r of T), columns 8 nt + 2 t4 + {0,1} (i = 16 Ic + ... of T)
#pragma unroll
                for (int nt = 0; nt < 2; ++nt)
#pragma unroll
                    for (int hf = 0; hf < 2; ++hf) {
                        uint32_t nl;
                        const uint32_t nh = split2(-y[nt][2 * hf], -y[nt][2 * hf + 1], nl);
                        const uint32_t so = blk(I, Ic) + (g8 + 8 * hf) * L::a_pitch + (8 * nt + 2 * t4) * 2;   // row-major U for the later products
                        *reinterpret_cast<uint32_t*>(ast + so) = nh;
                        *reinterpret_cast<uint32_t*>(ast + L::a_term_bytes + so) = nl;
                        const uint32_t j = 16 * I + g8 + 8 * hf;
                        const uint32_t off = (2 * Ic + nt) * L::op_sbo + (j >> 3) * 128 + (j & 7) * 16 + 4 * t4;
                        *reinterpret_cast<uint32_t*>(tbase + off) = nh;
                        *reinterpret_cast<uint32_t*>(tbase + L::t_term_bytes + off) = nl;
                    }
                __syncwarp();
            }
            GSEG(6);
            fence_proxy_async_smem();       // this warp's part of T: generic-proxy writes -> visible to the bulk copies
            tc_fence_before_sync();         // (and its reads of G are ordered before the next chunk's G MMAs)
            if (I == 0) cp_async_wait_all();   // the next owned chunk's raw gate values have landed
            named_bar_sync(1, 128);         // all of T(c) is in the staging buffer; G and the staging matrix may be reused
            GSEG(5);
            if (I == 0 && lane == 0) {
                if (c + csz < n_chunks) load_k(c + csz);
                mbar_arrive(&bars[direct ? BI.t_full : BI.t_staged]);   // the push warp takes it from here: these warps go on with the next owned chunk
            }
            __syncwarp();
            GSEG(2);
        }
    } else if (warp >= 12 && warp < 16) {
        // ================= R / W warps: R = beta (V - Gamma X) -> operand;  Wm -> [Wm_hi | Wm_lo] and W~ operands =================
        const int ra = 16 * q + g8, rb = ra + 8;
        const uint32_t op_a = (ra >> 3) * 128 + (ra & 7) * 16 + 4 * t4, op_b = (rb >> 3) * 128 + (rb & 7) * 16 + 4 * t4;
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t vi = c % NV, sb = c & 1, bt = c / kGCPB, gslot = bt & 1;
            if ((c % kGCPB) == 0) GW_(0, mbar_wait(&bars[BI.g_full + gslot], (bt >> 1) & 1));
            const float* b2 = gate + gslot * 3 * kGBatch + (c % kGCPB) * kGC;
            const float* eb = b2 + kGBatch;
            const float* be = b2 + 2 * kGBatch;
            const float ga = eb[ra], gb = eb[rb], bea = be[ra], beb = be[rb];
            const float b_last = b2[kGC - 1];
            const float la = ex2(b_last - b2[ra]), lb = ex2(b_last - b2[rb]);
            GW_(1, mbar_wait(&bars[BI.v_full + vi], (c / NV) & 1));
            const uint8_t* vs = sm + L::v_off + vi * L::v_bytes;
            uint32_t va[2], vb[2];
#pragma unroll
            for (int jb = 0; jb < 2; ++jb) {   // undo the 32-byte TMA swizzle: 16-byte chunk index ^= bit 7 of the address
                va[jb] = *reinterpret_cast<const uint32_t*>(vs + ra * 32 + ((jb ^ ((ra >> 2) & 1)) * 16) + 4 * t4);
                vb[jb] = *reinterpret_cast<const uint32_t*>(vs + rb * 32 + ((jb ^ ((rb >> 2) & 1)) * 16) + 4 * t4);
            }
            GW_(2, mbar_wait(&bars[BI.x_done], c & 1));
            tc_fence_after_sync();
            uint32_t xh[8], xl[8];
            tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_x), xh);
            tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_x + W), xl);
            tmem_ld_wait();
            tc_fence_before_sync();
            uint8_t* rop = sm + L::r_off;
#pragma unroll
            for (int jb = 0; jb < 2; ++jb) {
                // (packed fp32: FADD2 / FFMA2 / FMUL2 on the pairs of columns)
                const float2 xa = fadd2(make_float2(__uint_as_float(xh[4 * jb + 0]), __uint_as_float(xh[4 * jb + 1])),
                                        make_float2(__uint_as_float(xl[4 * jb + 0]), __uint_as_float(xl[4 * jb + 1])));
                const float2 xb = fadd2(make_float2(__uint_as_float(xh[4 * jb + 2]), __uint_as_float(xh[4 * jb + 3])),
                                        make_float2(__uint_as_float(xl[4 * jb + 2]), __uint_as_float(xl[4 * jb + 3])));
                const float2 ra2 = fmul2(make_float2(bea, bea), ffma2(make_float2(-ga, -ga), xa, make_float2(__uint_as_float(va[jb] << 16), __uint_as_float(va[jb] & 0xFFFF0000u))));
                const float2 rb2 = fmul2(make_float2(beb, beb), ffma2(make_float2(-gb, -gb), xb, make_float2(__uint_as_float(vb[jb] << 16), __uint_as_float(vb[jb] & 0xFFFF0000u))));
                const float r0 = ra2.x, r1 = ra2.y, r2 = rb2.x, r3 = rb2.y;
                uint32_t lo0, lo1;
                const uint32_t hi0 = split2(r0, r1, lo0), hi1 = split2(r2, r3, lo1);
                *reinterpret_cast<uint32_t*>(rop + jb * L::op_sbo + op_a) = hi0;
                *reinterpret_cast<uint32_t*>(rop + (jb + 2) * L::op_sbo + op_a) = lo0;
                *reinterpret_cast<uint32_t*>(rop + jb * L::op_sbo + op_b) = hi1;
                *reinterpret_cast<uint32_t*>(rop + (jb + 2) * L::op_sbo + op_b) = lo1;
            }
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bars[BI.r_full]);
                mbar_arrive(&bars[BI.x_read]);       // (X and the V tile were read before the operand was written)
                mbar_arrive(&bars[BI.v_read + vi]);
            }
            // ---- Wm ----
            GW_(3, mbar_wait(&bars[BI.w_done + sb], (c >> 1) & 1));
            tc_fence_after_sync();
            uint32_t wa[8], wb[8];
            tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_w), wa);
            tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_w + W), wb);
            tmem_ld_wait();
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BI.w_read]);
            if (c >= 1) GW_(4, mbar_wait(&bars[BI.u_done + ((c - 1) & 1)], ((c - 1) >> 1) & 1));   // U(c - 1) has read the W~ operand
            uint8_t* wv = sm + L::wv_off + sb * L::op_bytes;
            uint8_t* wt = sm + L::wt_off;
            // the decayed W~ operand first: it is the one on the carry chain (U waits for it); the Wm operand of the outputs after it
            float2 wA[2], wB[2];
#pragma unroll
            for (int jb = 0; jb < 2; ++jb) {
                wA[jb] = fadd2(make_float2(__uint_as_float(wa[4 * jb + 0]), __uint_as_float(wa[4 * jb + 1])),
                               make_float2(__uint_as_float(wb[4 * jb + 0]), __uint_as_float(wb[4 * jb + 1])));
                wB[jb] = fadd2(make_float2(__uint_as_float(wa[4 * jb + 2]), __uint_as_float(wa[4 * jb + 3])),
                               make_float2(__uint_as_float(wb[4 * jb + 2]), __uint_as_float(wb[4 * jb + 3])));
                const float2 sA = fmul2(make_float2(la, la), wA[jb]), sB = fmul2(make_float2(lb, lb), wB[jb]);
                uint32_t lo0, lo1;
                const uint32_t hi0 = split2(sA.x, sA.y, lo0), hi1 = split2(sB.x, sB.y, lo1);
                *reinterpret_cast<uint32_t*>(wt + jb * L::op_sbo + op_a) = hi0;
                *reinterpret_cast<uint32_t*>(wt + (jb + 2) * L::op_sbo + op_a) = lo0;
                *reinterpret_cast<uint32_t*>(wt + jb * L::op_sbo + op_b) = hi1;
                *reinterpret_cast<uint32_t*>(wt + (jb + 2) * L::op_sbo + op_b) = lo1;
            }
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BI.wt_full]);
            if (c >= 2) GW_(5, mbar_wait(&bars[BI.o2_done + sb], ((c - 2) >> 1) & 1));             // O2(c - 2) has read Wm operand sb
#pragma unroll
            for (int jb = 0; jb < 2; ++jb) {
                uint32_t lo0, lo1;
                const uint32_t hi0 = split2(wA[jb].x, wA[jb].y, lo0), hi1 = split2(wB[jb].x, wB[jb].y, lo1);
                *reinterpret_cast<uint32_t*>(wv + jb * L::op_sbo + op_a) = hi0;
                *reinterpret_cast<uint32_t*>(wv + (jb + 2) * L::op_sbo + op_a) = lo0;
                *reinterpret_cast<uint32_t*>(wv + jb * L::op_sbo + op_b) = hi1;
                *reinterpret_cast<uint32_t*>(wv + (jb + 2) * L::op_sbo + op_b) = lo1;
            }
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bars[BI.wv_full + sb]);
                if ((c % kGCPB) == (uint32_t)kGCPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
            }
        }
    } else if (warp >= 16 && warp < 20) {
        // ================= score warps: A^q = P (.) 2^(b_i - b_j) (j <= i), bf16 hi | lo, IN PLACE in TMEM =================
        const int ra = 16 * q + g8, rb = ra + 8;
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t pb = c & 1, bt = c / kGCPB, gslot = bt & 1;
            if ((c % kGCPB) == 0) GW_(0, mbar_wait_relaxed(&bars[BI.g_full + gslot], (bt >> 1) & 1));
            const float* b2 = gate + gslot * 3 * kGBatch + (c % kGCPB) * kGC;
            const float bia = b2[ra], bib = b2[rb];
            GW_(1, mbar_wait_relaxed(&bars[BI.p_done + pb], (c >> 1) & 1));
            tc_fence_after_sync();
            const uint32_t base = tmem_addr(tb, 32 * q, L::tm_p + pb * kGC);
#pragma unroll 1
            for (int ks = 0; ks < 4; ++ks) {
                uint32_t hi[4], lo[4];   // {row a block 0, row b block 0, row a block 1, row b block 1}: the 16x128b.x2 fragment
                if (ks <= q) {
                    uint32_t r[8];
                    tmem_ld_16x256b_x2(base + 16 * ks, r);
                    tmem_ld_wait();
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        const int j0 = 16 * ks + 8 * j + 2 * t4;
                        const float2 bj = *reinterpret_cast<const float2*>(b2 + j0);
                        float a0 = __uint_as_float(r[4 * j + 0]) * ex2(bia - bj.x);
                        float a1 = __uint_as_float(r[4 * j + 1]) * ex2(bia - bj.y);
                        float c0 = __uint_as_float(r[4 * j + 2]) * ex2(bib - bj.x);
                        float c1 = __uint_as_float(r[4 * j + 3]) * ex2(bib - bj.y);
                        // causal mask j <= i (only the diagonal step ks == q has anything to mask)
                        a0 = (j0 <= ra) ? a0 : 0.f;
                        a1 = (j0 + 1 <= ra) ? a1 : 0.f;
                        c0 = (j0 <= rb) ? c0 : 0.f;
                        c1 = (j0 + 1 <= rb) ? c1 : 0.f;
                        hi[2 * j] = split2(a0, a1, lo[2 * j]);
                        hi[2 * j + 1] = split2(c0, c1, lo[2 * j + 1]);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < 4; ++i) hi[i] = lo[i] = 0u;
                }
                tmem_st_16x128b_x2(base + 16 * ks, hi);
                tmem_st_16x128b_x2(base + 16 * ks + 8, lo);
            }
            tmem_st_wait();
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bars[BI.a_full + pb]);
                if ((c % kGCPB) == (uint32_t)kGCPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
            }
        }
    } else if (warp >= 20 && warp < 24) {
        // ================= epilogue warps: o_i = 2^(b_i) (Yh_i + Yl_i) + O2_i =================
        const int ra = 16 * q + g8, rb = ra + 8;
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t pb = c & 1, bt = c / kGCPB, gslot = bt & 1;
            if ((c % kGCPB) == 0) GW_(0, mbar_wait_relaxed(&bars[BI.g_full + gslot], (bt >> 1) & 1));
            const float* eb = gate + gslot * 3 * kGBatch + kGBatch + (c % kGCPB) * kGC;
            const float ea = eb[ra], ebb = eb[rb];
            GW_(1, mbar_wait_relaxed(&bars[BI.y_done + pb], (c >> 1) & 1));
            tc_fence_after_sync();
            float y[8];
            {
                uint32_t yh[8], yl[8];
                tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_y + pb * 2 * W), yh);
                tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_y + pb * 2 * W + W), yl);
                tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 8; ++i) y[i] = __uint_as_float(yh[i]) + __uint_as_float(yl[i]);
            }
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bars[BI.y_free + pb]);
                if ((c % kGCPB) == (uint32_t)kGCPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
            }
            GW_(2, mbar_wait_relaxed(&bars[BI.o2_done + pb], (c >> 1) & 1));
            tc_fence_after_sync();
            uint32_t oa[8], ob[8];
            tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_o2 + pb * 2 * W), oa);
            tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q, L::tm_o2 + pb * 2 * W + W), ob);
            tmem_ld_wait();
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BI.o2_free + pb]);
            const uint64_t t0 = (uint64_t)c * kGC;
            const int n = (int)((T - t0) < (uint64_t)kGC ? (T - t0) : (uint64_t)kGC);
            float* pa = o + (((size_t)b * t_stride + t0 + ra) * H + h) * DV + dv0 + 2 * t4;
            float* pc = o + (((size_t)b * t_stride + t0 + rb) * H + h) * DV + dv0 + 2 * t4;
#pragma unroll
            for (int jb = 0; jb < 2; ++jb) {
                if (ra < n)
                    *reinterpret_cast<float2*>(pa + 8 * jb) =
                        make_float2(fmaf(ea, y[4 * jb + 0], __uint_as_float(oa[4 * jb + 0]) + __uint_as_float(ob[4 * jb + 0])),
                                    fmaf(ea, y[4 * jb + 1], __uint_as_float(oa[4 * jb + 1]) + __uint_as_float(ob[4 * jb + 1])));
                if (rb < n)
                    *reinterpret_cast<float2*>(pc + 8 * jb) =
                        make_float2(fmaf(ebb, y[4 * jb + 2], __uint_as_float(oa[4 * jb + 2]) + __uint_as_float(ob[4 * jb + 2])),
                                    fmaf(ebb, y[4 * jb + 3], __uint_as_float(oa[4 * jb + 3]) + __uint_as_float(ob[4 * jb + 3])));
            }
        }
    } else if (warp >= 24 && warp < 28) {
        // ================= state warps: the carry  S <- 2^(b_C) S + (Uh + Ul), fp32 FMA in registers =================
        // fragment layout and the stmatrix transposition into the K-major S^T operand as in scan_kernel.cu
        constexpr int NLG = (DK == 128) ? 2 : 1;
        const uint32_t kq = (DK == 128) ? 32 * q : 16 * q;
        float S[NLG][2][4];
#pragma unroll
        for (int lg = 0; lg < NLG; ++lg)
#pragma unroll
            for (int jb = 0; jb < 2; ++jb)
#pragma unroll
                for (int hl = 0; hl < 2; ++hl) {
                    float2 x = make_float2(0.f, 0.f);
                    if (state_in) x = *reinterpret_cast<const float2*>(state_in + ((size_t)bh * DK + kq + 16 * lg + 8 * hl + g8) * DV + dv0 + 8 * jb + 2 * t4);
                    S[lg][jb][2 * hl] = x.x;
                    S[lg][jb][2 * hl + 1] = x.y;
                }
        // stmatrix row addresses: lane L supplies row L % 8 (column n of S) of matrix L / 8 = {hi k 0-7, hi k 8-15, lo k 0-7, lo k 8-15}
        // of the (lg, jb) block; operand row R = 16 term + 8 jb + n, 16-byte chunk ((k0 % 64) / 8) ^ (R % 8)
        uint32_t st_off[NLG][2];
#pragma unroll
        for (int lg = 0; lg < NLG; ++lg)
#pragma unroll
            for (int jb = 0; jb < 2; ++jb) {
                const uint32_t term = lane >> 4, hl = (lane >> 3) & 1, n = lane & 7;
                const uint32_t R = term * W + 8 * jb + n, k0 = kq + 16 * lg + 8 * hl;
                st_off[lg][jb] = (k0 >> 6) * L::s_half_bytes + R * 128 + ((((k0 & 63) >> 3) ^ (R & 7)) << 4);
            }
        auto write_s_operand = [&](uint32_t sb) {
            const uint32_t base = sm_a + L::s_off + sb * L::s_bytes;
#pragma unroll
            for (int lg = 0; lg < NLG; ++lg)
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {
                    uint32_t lo0, lo1;
                    const uint32_t hi0 = split2(S[lg][jb][0], S[lg][jb][1], lo0), hi1 = split2(S[lg][jb][2], S[lg][jb][3], lo1);
                    stmatrix_x4_trans(base + st_off[lg][jb], hi0, hi1, lo0, lo1);
                }
        };
        write_s_operand(0);
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars[BI.s_full]);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t ub = c & 1, bt = c / kGCPB, gslot = bt & 1;
            if ((c % kGCPB) == 0) GW_(0, mbar_wait(&bars[BI.g_full + gslot], (bt >> 1) & 1));
            const float gam = gate[gslot * 3 * kGBatch + kGBatch + (c % kGCPB) * kGC + kGC - 1];
            GW_(1, mbar_wait(&bars[BI.u_done + ub], (c >> 1) & 1));
            tc_fence_after_sync();
            uint32_t uh[NLG][8], ul[NLG][8];
#pragma unroll
            for (int lg = 0; lg < NLG; ++lg) {
                tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q + 16 * lg, L::tm_u + ub * 2 * W), uh[lg]);
                tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q + 16 * lg, L::tm_u + ub * 2 * W + W), ul[lg]);
            }
            tmem_ld_wait();
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bars[BI.u_empty + ub]);
                if ((c % kGCPB) == (uint32_t)kGCPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
            }
#pragma unroll
            for (int lg = 0; lg < NLG; ++lg)
#pragma unroll
                for (int jb = 0; jb < 2; ++jb)
#pragma unroll
                    for (int e = 0; e < 4; e += 2) {
                        const float2 u = fadd2(make_float2(__uint_as_float(uh[lg][4 * jb + e]), __uint_as_float(uh[lg][4 * jb + e + 1])),
                                               make_float2(__uint_as_float(ul[lg][4 * jb + e]), __uint_as_float(ul[lg][4 * jb + e + 1])));
                        const float2 sn = ffma2(make_float2(gam, gam), make_float2(S[lg][jb][e], S[lg][jb][e + 1]), u);
                        S[lg][jb][e] = sn.x;
                        S[lg][jb][e + 1] = sn.y;
                    }
            if (c + 1 < n_chunks) {
                // operand buffer (c + 1) % 2 was last read by X(c - 1), Y(c - 1): complete, they were issued before U(c) by the same thread
                write_s_operand((c + 1) & 1);
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars[BI.s_full + ((c + 1) & 1)]);
            }
        }
#pragma unroll
        for (int lg = 0; lg < NLG; ++lg)
#pragma unroll
            for (int jb = 0; jb < 2; ++jb)
#pragma unroll
                for (int hl = 0; hl < 2; ++hl)
                    *reinterpret_cast<float2*>(state_out + ((size_t)bh * DK + kq + 16 * lg + 8 * hl + g8) * DV + dv0 + 8 * jb + 2 * t4) =
                        make_float2(S[lg][jb][2 * hl], S[lg][jb][2 * hl + 1]);
    }

    GPROF_END;
    // ---- teardown: the state and epilogue warps have waited on the last commits of every MMA group but G / P, whose results the
    // T and score warps have read ----
    tc_fence_before_sync();
    cluster_sync();   // no peer still copies into this CTA or arrives on its barriers
    if (warp == 2) tmem_dealloc(tb, L::tmem_cols);
}

template <int DK>
static int launch_gdn_t(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* beta,
                 const float* state_in, float* state_out, float* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    using L = GdnCfg<DK>;
    const int rc0 = ensure_dyn_smem(ctx, kSlotGdn + (DK == 128 ? 0 : 1), esc_gdn_scan_kernel<DK>, (int)L::total);
    if (rc0 != ESC_OK) return rc0;
    if (!state_out) return ESC_OK;   // prepare-only call (before a stream capture)
    CUtensorMap tq, tk, tv;
    const void* qq = T ? q : (const void*)state_out;   // T == 0: the maps are never dereferenced, any valid address will do
    const void* kk = T ? k : (const void*)state_out;
    const void* vv = T ? v : (const void*)state_out;
    const uint64_t ts = t_stride ? t_stride : 1;
    int rc = make_tmap_halves(&tq, qq, DK, s.H, T, ts, s.B, kGC);
    if (rc == ESC_OK) rc = make_tmap_halves(&tk, kk, DK, s.H, T, ts, s.B, kGC);
    if (rc == ESC_OK) rc = make_tmap(&tv, vv, s.dv, s.H, T, ts, s.B, kGW, kGC, CU_TENSOR_MAP_SWIZZLE_32B);
    if (rc != ESC_OK) return rc;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(s.dv / kGW, s.B * s.H);   // the d_v slices of a (b, h) are one cluster (4 or 8 CTAs): they share the chunk inverses
    cfg.blockDim = dim3(L::kThreads);
    cfg.dynamicSmemBytes = L::total;
    cfg.stream = stream;
    cudaLaunchAttribute attr[2];
    memset(attr, 0, sizeof attr);
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = T <= kGdnShortT ? 1 : kGdnCluster;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddepcontrol.* in the kernel
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 2;
    ESC_CUDA(cudaLaunchKernelEx(&cfg, esc_gdn_scan_kernel<DK>, tq, tk, tv, g, beta, state_in, state_out, o, s.H, s.dv, T, t_stride));
    return ESC_OK;
}

#ifdef ESC_GDN_PROF
extern "C" int esc_debug_gdn_prof_read(long long* host) { return (int)cudaMemcpyFromSymbol(host, g_gdn_prof, sizeof(g_gdn_prof)); }
#endif

int launch_gdn_mma(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* beta,
                   const float* state_in, float* state_out, float* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    if (s.dv % kGW || (s.dv / kGW) % kGdnCluster) return ESC_ERR_UNSUPPORTED;
    if (s.dk == 128) return launch_gdn_t<128>(ctx, s, q, k, v, g, beta, state_in, state_out, o, T, t_stride, stream);
    if (s.dk == 64) return launch_gdn_t<64>(ctx, s, q, k, v, g, beta, state_in, state_out, o, T, t_stride, stream);
    return ESC_ERR_UNSUPPORTED;
}

}  // namespace esc
