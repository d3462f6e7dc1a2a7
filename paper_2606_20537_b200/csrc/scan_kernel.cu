// Chunked gated linear-attention scan, sm_100a tensor-core path (include/esc.h: esc_linattn_scan).
//
// Definition (BASELINE.json north_star; "a fold over the entire prefix", folded "per
// chunk" PAPER.md:169):   S_t = g_t S_{t-1} + k_t^T v_t ,  o_t = q_t S_t.
// Chunk algebra (exact-arithmetic equivalent; every exponent <= 0), 64-token chunks, b_i = sum_{r<=i} log2 g_r:
//     [P | O1] = Q [K^T | S_hi | S_lo]                (64 x (64 + 2W))   ONE tcgen05.mma group  M=64 N=64+2W K=d_k   (SS)
//     A_ij     = P_ij 2^(b_i - b_j) [j <= i]          fp32 ALU + MUFU, split into bf16 hi + lo, written back IN PLACE into
//                                                      the TMEM columns P came from (tcgen05.st)
//     O2       = A_hi V + A_lo V                      (64 x W)           tcgen05.mma  M=64 N=W K=64, A operand FROM TMEM (TS)
//     o_i      = 2^(b_i) (O1h_i + O1l_i) + O2_i       fp32 epilogue
//     U        = K^T [V~_hi | V~_lo] , V~_j = 2^(b_C - b_j) v_j   (d_k x 2W)  tcgen05.mma  M=d_k N=2W K=64   (SS)
//     S_next   = 2^(b_C) S_prev + (Uh + Ul)           fp32 FMA in registers (the carry chain)
//
// Decomposition.  The columns of S are independent: one CTA owns (b, h, W columns of d_v) and walks the chunks in order with
// its [d_k x W] state slice in registers.  W (16 or 32) is a function of the SHAPE KEY only (scan_tile_columns: the widest
// tile that still gives every SM a CTA), never of T, so a cold run and a restore-then-continue run of one key execute the
// same arithmetic.  Up to four neighbouring d_v slices of a head form a thread-block cluster for ONE
// purpose: the Q and K tiles are loaded once per cluster (CTA r loads rows [16r, 16r+16) of each and TMA-multicasts them to
// all), which divides the L2 -> SM traffic of the shared operands by the cluster size.  Everything else is CTA-local.
//
// What this layout is for (r01 measured the previous design at 1400 cycles per chunk per CTA, bound by shared-memory
// bandwidth: ~160 KB of operand reads, TMA writes, score exchange and operand staging per chunk): every byte that does not have
// to cross shared memory does not.
//   * P and O1 share their A operand (Q): one MMA group with the K tile and the transposed state operand S^T stacked along N
//     reads Q once per chunk instead of twice.  S^T lives directly under the K tile in the stage ([K rows | S_hi^T | S_lo^T],
//     K-major, 128-byte swizzle), written there by the state warps.
//   * The score matrix never touches shared memory: the score warps read P from TMEM, form A = P (.) D in registers and store
//     its bf16 hi / lo terms back into the same TMEM columns (a 64-key row of fp32 P is exactly a row of hi|lo bf16 pairs);
//     O2 takes its A operand from TMEM.  No A buffers, no slice exchange between CTAs, no cluster barrier per chunk.
//   * O2 reads V straight from a small ring of V tiles of its own (6 deep), so the score path never holds a Q/K stage.
// Per chunk and CTA (d_k = 128): 20 tcgen05.mma (8 + 4 + 8), 3 + 1 + 3 commits; shared-memory traffic ~114 KB at W = 16,
// ~148 KB at W = 32 (vs ~160 KB for 16 columns before).
//
// Warp roles (mbarrier-synchronised software pipeline, no CTA-wide barrier in the loop):
//   warp 0         TMA producer (Q/K row slices multicast to the cluster, own V tile; L2 prefetch ahead)
//   warp 1         gate warp: log2 g, segmented warp-shuffle prefix sums, 256 tokens per batch
//   warp 2         issuer of [P | O1]      warp 3   issuer of U      last warp   issuer of O2
//   warps 4-7      V~ warps: V -> V~ hi/lo operand (own barriers: U and the carry never wait for the scores)
//   warps 8-15     score warps (two per TMEM lane quadrant, two 16-key steps each): P (TMEM) -> A hi|lo (TMEM), in place
//   warps 16-19    epilogue warps: O1, O2 (TMEM) -> o (global)
//   warps 20-23    state warps (W = 32: 20-27, 16 columns each): U (TMEM) -> carry S in fp32 registers -> S^T operand
//
// Bit-identity: the carry is a pure function of (S_prev bits, chunk inputs); there is no T-dependent
// tiling, no atomics, no split-K; every accumulator is produced by ONE issuer thread in a fixed order, every A element by
// one thread.  Calls of up to kShortT tokens launch the same kernel without the cluster (whole-tile TMA loads instead of
// multicast row slices): the arithmetic is the same instruction for instruction.  Precision: raw Q, K, V are
// the bf16 inputs; A, V~, S_prev are two-term bf16 splits (hi + lo).
#include <cuda.h>
#include <cuda_bf16.h>

#include "esc_internal.h"
#include "sm100_ptx.cuh"
#include "tmap.h"

namespace esc {

using namespace ptx;
typedef __nv_bfloat16 bf16;

constexpr int kC = 64;             // token tile (the key's chunk, 64 or 128, is a multiple of it)
constexpr int kGateBatch = 256;    // tokens per gate-warp batch
constexpr int kCPB = kGateBatch / kC;
constexpr int kPrefetchAhead = 6;  // chunks the producer prefetches into L2 ahead of its smem ring
constexpr int kVtThreads = 128;    // threads of the four V~ warps

#ifdef ESC_TC_TRACE   // bring-up only: per-chunk clock64() stamps of CTA (0,0), read back with esc_debug_trace_read
__device__ long long g_tc_trace[16 * 64];
#define TC_TRACE(ev, c) do { if (blockIdx.x == 0 && blockIdx.y == 0 && (c) < 64) g_tc_trace[(ev) * 64 + (c)] = clock64(); } while (0)
#else
#define TC_TRACE(ev, c) do { } while (0)
#endif

#ifdef ESC_SCAN_PROF   // bring-up only: cycles every role of CTA (0,0) spends in each of its waits, and in its loop in total
__device__ long long g_scan_prof[32 * 8];
#define PROF_DECL long long prof_[8] = {0, 0, 0, 0, 0, 0, 0, 0}; const long long prof_t0_ = clock64();
#define PW(slot, call) do { const long long t_ = clock64(); call; prof_[slot] += clock64() - t_; } while (0)
#define PROF_END do { if (blockIdx.x == 0 && blockIdx.y == 0 && lane == 0) { prof_[7] = clock64() - prof_t0_; \
        for (int i_ = 0; i_ < 8; ++i_) g_scan_prof[warp * 8 + i_] = prof_[i_]; } } while (0)
#else
#define PROF_DECL
#define PW(slot, call) call
#define PROF_END do { } while (0)
#endif

template <int DK, int W, int CS>
struct ScanCfg {
    static constexpr int NH = DK / 64;                         // 64-column halves of a Q / K tile
    static constexpr int NS = (W == 16) ? 4 : 3;               // Q | K+S^T stages
    static constexpr int NV = 6;                               // V tiles
    static constexpr int NB = (W == 16) ? 4 : 3;               // [P/A | O1] accumulator buffers (TMEM)
    static constexpr int NUB = (W == 16) ? 2 : 1;              // U accumulator buffers (W = 32: one, the columns go to the third [P|O1] buffer)
    static constexpr int NVT = (W == 16) ? 3 : 2;              // V~ operand buffers
    static constexpr int NSW = W / 16;                         // state-warp sets (16 columns of the slice each)
    static constexpr int kWarps = 20 + 4 * NSW + 1;
    static constexpr int kThreads = kWarps * 32;
    static constexpr int kO2Warp = kWarps - 1;
    static constexpr int NPO = kC + 2 * W;                     // N of the merged MMA = TMEM columns of one accumulator buffer
    static constexpr uint32_t q_half_bytes = kC * 128;         // one [64 x 64] bf16 half tile of Q
    static constexpr uint32_t q_bytes = NH * q_half_bytes;
    static constexpr uint32_t ks_half_bytes = NPO * 128;       // [K rows 0..63 | S_hi^T rows | S_lo^T rows] x 64 columns of d_k
    static constexpr uint32_t ks_bytes = NH * ks_half_bytes;
    static constexpr uint32_t k_tile_bytes = NH * kC * 128;    // what TMA writes into the K rows
    static constexpr uint32_t stage_bytes = q_bytes + ks_bytes;
    static constexpr uint32_t v_bytes = kC * W * 2;            // [64 x W] bf16, swizzle = row width (32 B / 64 B)
    static constexpr uint32_t sbo_vt = (kC / 8) * 128;         // V~ operand: 8-column groups of [64 tokens x 8] bf16
    static constexpr uint32_t vt_bytes = (2 * W / 8) * sbo_vt;
    static constexpr uint32_t stage_off = 0;
    static constexpr uint32_t v_off = stage_off + NS * stage_bytes;
    static constexpr uint32_t vt_off = v_off + NV * v_bytes;
    static constexpr uint32_t gate_off = vt_off + NVT * vt_bytes;   // [2][b2[256], eb[256]] fp32
    static constexpr uint32_t bar_off = gate_off + 2 * 2 * kGateBatch * 4;
    static constexpr int NU = 4;                               // ring of "U(c) done" barriers (> NVT: the V~ warps wait on chunk c - NVT's)
    static constexpr uint32_t n_bars = 3 * NS + 3 * NV + 3 * NB + NVT + NU + 8;   // (u_empty has two slots whatever NUB)
    static constexpr uint32_t total = bar_off + 64 * 8 + 16 + 1024;   // + alignment slack
    // TMEM columns
    static constexpr uint32_t tm_po = 0;                       // [NB] x NPO: P -> A (columns 0..63), O1 hi | lo (64..64+2W)
    static constexpr uint32_t tm_o2 = NB * NPO;                // [2] x W
    static constexpr uint32_t tm_u = tm_o2 + 2 * W;            // [NUB] x 2W
    static constexpr uint32_t tmem_cols = 512;
    static_assert(tm_u + NUB * 2 * W <= tmem_cols, "TMEM budget");
    static_assert(stage_bytes % 1024 == 0 && q_bytes % 1024 == 0 && ks_half_bytes % 1024 == 0, "128B-swizzled regions need 1024-byte alignment");
    static_assert(v_bytes % 1024 == 0 && v_off % 1024 == 0, "V tiles keep their swizzle alignment");
    static_assert(n_bars <= 64, "barrier area");
    static_assert(total <= 232448, "shared memory budget");
    static_assert(W == 16 || W == 32, "d_v tile");
    static_assert(kThreads <= 1024, "block size");
};

// One tcgen05.commit costs its issuing thread about as much as an MMA, so every MMA group commits ONCE to a ring of "done"
// barriers and everybody who cares about that event waits on the ring entry (a wait on a completed barrier is cheap):
//   o2_done[c % NV]: O2(c) has completed -> the epilogue (o is ready), the producer (V tile c % NV, together with v_read: the V~
//                    warps have read it), the [P|O1] issuer (accumulator c % NB, together with po_read: the epilogue has read O1)
//   u_done[c % NU]:  U(c) has completed  -> the state warps (U is ready), the V~ warps (operand buffer of chunk c + NVT)
// A waiter is never more than one phase behind a ring entry (see the parity notes at the waits).
struct ScanBars {   // indices into the mbarrier array
    int full, empty, s_full, v_full, v_read, o2_done, po_full, po_read, a_full, vt_full, u_done, o2_empty, u_empty, g_full, g_empty;
};
template <int DK, int W, int CS>
__device__ __forceinline__ constexpr ScanBars scan_bars() {
    using L = ScanCfg<DK, W, CS>;
    ScanBars b{};
    int i = 0;
    b.full = i; i += L::NS;
    b.empty = i; i += L::NS;
    b.s_full = i; i += L::NS;
    b.v_full = i; i += L::NV;
    b.v_read = i; i += L::NV;
    b.o2_done = i; i += L::NV;
    b.po_full = i; i += L::NB;
    b.po_read = i; i += L::NB;
    b.a_full = i; i += L::NB;
    b.vt_full = i; i += L::NVT;
    b.u_done = i; i += L::NU;
    b.o2_empty = i; i += 2;
    b.u_empty = i; i += 2;
    b.g_full = i; i += 2;
    b.g_empty = i; i += 2;
    return b;
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

template <int DK, int W, int CS, typename OutT>
__global__ void __launch_bounds__(ScanCfg<DK, W, CS>::kThreads, 1)
esc_scan_kernel(const __grid_constant__ CUtensorMap tq, const __grid_constant__ CUtensorMap tk,
                const __grid_constant__ CUtensorMap tv, const __grid_constant__ CUtensorMap tqp, const __grid_constant__ CUtensorMap tkp,
                const float* __restrict__ g, const float* state_in,
                float* state_out, OutT* __restrict__ o, uint32_t H, uint32_t DV, uint64_t T, uint64_t t_stride) {
    using L = ScanCfg<DK, W, CS>;
    constexpr ScanBars BI = scan_bars<DK, W, CS>();
    constexpr int NS = L::NS, NV = L::NV, NB = L::NB, NVT = L::NVT, NSW = L::NSW, NPO = L::NPO, NU = L::NU, NUB = L::NUB;
    constexpr int NR = kC / CS;                     // Q / K rows this CTA loads (and multicasts)
    constexpr uint16_t kAll = (uint16_t)((1u << CS) - 1);

    extern __shared__ uint8_t smem_raw[];
    uint8_t* sm = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // same offset in every CTA of the cluster
    const uint32_t sm_a = smem_u32(sm);
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + L::bar_off);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sm + L::bar_off + 64 * 8);
    float* gate = reinterpret_cast<float*>(sm + L::gate_off);   // [2][2][256]: b2 then eb per slot

    // (the shuffle tells the compiler that the warp index is warp-uniform: the role branches become uniform branches, and inside
    // them descriptors, barrier addresses and loop state live in uniform registers instead of being moved there before every MMA)
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    uint32_t rank = 0;
    if constexpr (CS > 1) rank = cluster_ctarank();   // clusters are CS consecutive d_v slices (blockIdx.x) of one (b, h)
    const uint32_t bh = blockIdx.y, b = bh / H, h = bh % H, dv0 = blockIdx.x * W;
    const uint32_t row0 = rank * NR;    // first Q / K row of this CTA's share of a tile
    const uint32_t n_chunks = (uint32_t)((T + kC - 1) / kC);
    const int q = warp & 3;   // TMEM lane quadrant this warp may access
    // Programmatic dependent launch: the next kernel of the stream / graph (typically the next layer's scan) may start
    // its on-chip setup while this one runs; everything this kernel reads from or writes to global memory comes after
    // griddepcontrol.wait below, i.e. after the preceding kernel has completed and flushed.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (threadIdx.x == 0) TC_TRACE(11, 0);

    // the waits of the roles that run ahead of the pipeline (producer, gate warp).  Long calls poll tightly: a back-off of 64 ns
    // in these waits costs them 1.5 % (r02: 0.329 -> 0.334 of roofline at B 1, 16k); the one-chunk launches of the suffix path
    // are faster WITH it (67.6 vs 69.6 us per 18 layers): fewer polls beside the few warps that have work.
    auto wait_ahead = [&](uint64_t* bar, uint32_t parity) {
        if constexpr (CS > 1) mbar_wait(bar, parity);
        else mbar_wait_relaxed(bar, parity);
    };
    // commit that every CTA of the cluster must see (stage reuse: every CTA writes into every CTA's stage)
    auto commit_all = [&](uint64_t* bar) {   // warp-uniform (every lane calls it, one elected lane issues)
        if constexpr (CS > 1) mma_commit_mc_w(bar, kAll);
        else mma_commit_w(bar);
    };

    // ---- one-time setup, on-chip part (under programmatic dependent launch it overlaps the preceding kernel) -----------
    if (warp == 0 && lane == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(&bars[BI.full + i], 1);
            mbar_init(&bars[BI.empty + i], 2 * CS);           // [P|O1] and U issuers of every CTA of the cluster
            mbar_init(&bars[BI.s_full + i], 4 * NSW);
        }
        for (int i = 0; i < NV; ++i) {
            mbar_init(&bars[BI.v_full + i], 1); mbar_init(&bars[BI.v_read + i], 4); mbar_init(&bars[BI.o2_done + i], 1);
        }
        for (int i = 0; i < NB; ++i) {
            mbar_init(&bars[BI.po_full + i], 1);
            mbar_init(&bars[BI.po_read + i], 4);              // the epilogue warps have read O1
            mbar_init(&bars[BI.a_full + i], 8);
        }
        for (int i = 0; i < NVT; ++i) mbar_init(&bars[BI.vt_full + i], 4);
        for (int i = 0; i < NU; ++i) mbar_init(&bars[BI.u_done + i], 1);
        for (int i = 0; i < 2; ++i) {
            mbar_init(&bars[BI.o2_empty + i], 4);
            mbar_init(&bars[BI.u_empty + i], 4 * NSW);
            mbar_init(&bars[BI.g_full + i], 1); mbar_init(&bars[BI.g_empty + i], 4 + 8 + 4 + 4 * NSW);
        }
        fence_mbar_init();
        tma_prefetch_desc(&tq); tma_prefetch_desc(&tk); tma_prefetch_desc(&tv); tma_prefetch_desc(&tqp); tma_prefetch_desc(&tkp);
    }
    if (warp == 2) tmem_alloc(tmem_slot, L::tmem_cols);
    tc_fence_before_sync();
    // every CTA's barriers are initialised before any peer multicasts into its stages or arrives on them
    if constexpr (CS > 1) cluster_sync();
    else __syncthreads();
    tc_fence_after_sync();
    const uint32_t tb = __shfl_sync(0xffffffffu, *tmem_slot, 0);
    if (threadIdx.x == 0) TC_TRACE(14, 0);
    asm volatile("griddepcontrol.wait;" ::: "memory");   // ---- global memory may be touched from here on ----
    if (threadIdx.x == 0) TC_TRACE(12, 0);
    PROF_DECL

    if (warp == 0) {
        // ================= TMA producer =================
        if (lane == 0) {
            // L2 prefetch of chunk c: the Q and K tiles are shared by the cluster, so CTA c % CS pulls both WHOLE tiles (one
            // instruction each through the 5-D halves map) and every CTA its own V tile: 1 + 2 / CS prefetch instructions per chunk
            // instead of 5 (an UTMAPF costs the producer ~90 cycles like any TMA instruction, r02 wait accounting)
            auto prefetch_chunk = [&](uint32_t c) {
                const int t0 = (int)(c * kC);
                if (CS == 1 || c % CS == rank) {
                    tma_prefetch_5d(&tqp, 0, t0, 0, (int)h, (int)b);
                    tma_prefetch_5d(&tkp, 0, t0, 0, (int)h, (int)b);
                }
                tma_prefetch_4d(&tv, (int)dv0, (int)h, t0, (int)b);
            };
            for (uint32_t c = NS; c < n_chunks && c < (uint32_t)(NS + kPrefetchAhead); ++c) prefetch_chunk(c);
            for (uint32_t c = 0; c < n_chunks; ++c) {
                if (c + NS + kPrefetchAhead < n_chunks) prefetch_chunk(c + NS + kPrefetchAhead);
                const uint32_t s = c % NS, vi = c % NV;
                const int t0 = (int)(c * kC);
                uint8_t* st = sm + L::stage_off + s * L::stage_bytes;
                // the stage is free once the [P|O1] and U issuers of all CS CTAs have committed chunk c - NS
                if (CS > 1 || c >= (uint32_t)NS) PW(0, wait_ahead(&bars[BI.empty + s], ((c / NS) & 1) ^ 1));   // (a short call's first round: fresh)
                uint64_t* full = &bars[BI.full + s];
                mbar_arrive_expect_tx(full, L::q_bytes + L::k_tile_bytes);   // arrives in CS row slices, one from each CTA
                if constexpr (CS > 1) {
#pragma unroll
                    for (int hh = 0; hh < L::NH; ++hh) {
                        tma_load_4d_mc(st + hh * L::q_half_bytes + row0 * 128, &tq, full, hh * 64, (int)h, t0 + (int)row0, (int)b, kAll);
                        tma_load_4d_mc(st + L::q_bytes + hh * L::ks_half_bytes + row0 * 128, &tk, full, hh * 64, (int)h, t0 + (int)row0,
                                       (int)b, kAll);
                    }
                } else {
                    // on its own a CTA takes the whole Q tile in one instruction: the map has the 64-column halves as its third
                    // dimension (d % 64, t, d / 64, h, b), so a box of (64, 64, NH) lands as [half][token][64]
                    tma_load_5d(st, &tq, full, 0, t0, 0, (int)h, (int)b);
#pragma unroll
                    for (int hh = 0; hh < L::NH; ++hh)
                        tma_load_4d(st + L::q_bytes + hh * L::ks_half_bytes, &tk, full, hh * 64, (int)h, t0, (int)b);
                }
                // V tiles have a ring of their own: O2 (the end of the score path) reads V from it, so a Q/K stage is
                // released as soon as [P|O1] and U are done with it
                if (CS > 1 || c >= (uint32_t)NV) {
                    PW(1, wait_ahead(&bars[BI.v_read + vi], ((c / NV) & 1) ^ 1));      // the V~ warps and O2 of chunk c - NV
                    PW(1, wait_ahead(&bars[BI.o2_done + vi], ((c / NV) & 1) ^ 1));     // are done with V tile vi
                }
                mbar_arrive_expect_tx(&bars[BI.v_full + vi], L::v_bytes);
                tma_load_4d(sm + L::v_off + vi * L::v_bytes, &tv, &bars[BI.v_full + vi], (int)dv0, (int)h, t0, (int)b);
                TC_TRACE(0, c);
            }
            // tail: every peer's last commits have reached this CTA's barriers before anyone may exit
            for (uint32_t c = n_chunks > (uint32_t)NS ? n_chunks - NS : 0; c < n_chunks; ++c)
                mbar_wait(&bars[BI.empty + c % NS], (c / NS) & 1);
        }
    } else if (warp == 1) {
        // ================= gate warp: b2_i = sum_{r<=i in chunk} log2 g_r, 256 tokens per batch =================
        const uint32_t n_batches = (uint32_t)((T + kGateBatch - 1) / kGateBatch);
        constexpr int GL = kC / 8;   // lanes per chunk
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
            if (CS > 1 || bt >= 2) PW(0, wait_ahead(&bars[BI.g_empty + slot], ((bt >> 1) & 1) ^ 1));
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
        // ================= issuer: [P | O1] = Q [K^T | S_hi | S_lo]  (B operand: the K tile with S^T stacked under it) =======
        // the whole warp runs the loop (warp-uniform operands), one elected lane issues each instruction
        constexpr uint32_t idPO = idesc_bf16(kC, NPO, 0, 0);
        const uint64_t dQ0 = smem_desc(sm_a + L::stage_off, 16, 1024, kSwz128);
        const uint64_t dB0 = smem_desc(sm_a + L::stage_off + L::q_bytes, 16, 1024, kSwz128);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t s = c % NS, pb = c % NB;
            PW(0, mbar_wait(&bars[BI.full + s], (c / NS) & 1));
            // accumulator pb is free once the epilogue has read O1(c - NB) and O2(c - NB) has read A.  The O2 issuer is never
            // ahead of this warp, so the ring entry of chunk c - NB cannot have moved on to a later phase.
            if (CS > 1 || c >= (uint32_t)NB) PW(1, mbar_wait(&bars[BI.po_read + pb], ((c / NB) & 1) ^ 1));
            if (c >= (uint32_t)NB) PW(1, mbar_wait(&bars[BI.o2_done + (c - NB) % NV], ((c - NB) / NV) & 1));
            PW(2, mbar_wait(&bars[BI.s_full + s], (c / NS) & 1));      // the carried state: last, it is the one on the chain
            tc_fence_after_sync();
            const uint64_t dQ = smem_desc_advance(dQ0, s * L::stage_bytes), dB = smem_desc_advance(dB0, s * L::stage_bytes);
            const uint32_t dD = tb + L::tm_po + pb * NPO;
#pragma unroll
            for (int ks = 0; ks < DK / 16; ++ks)
                mma_bf16_ss_w(dD, smem_desc_advance(dQ, (ks / 4) * L::q_half_bytes + (ks % 4) * 32),
                              smem_desc_advance(dB, (ks / 4) * L::ks_half_bytes + (ks % 4) * 32), idPO, ks > 0);
            mma_commit_w(&bars[BI.po_full + pb]);
            commit_all(&bars[BI.empty + s]);
            if (lane == 0) TC_TRACE(1, c);
        }
    } else if (warp == 3) {
        // ================= issuer: U = K^T [V~_hi | V~_lo] (A operand = the K rows of the stage read MN-major) =================
        constexpr uint32_t idU = idesc_bf16(DK, 2 * W, 1, 1);
        const uint64_t dK0 = smem_desc(sm_a + L::stage_off + L::q_bytes, L::ks_half_bytes, 1024, kSwz128);
        const uint64_t dV0 = smem_desc(sm_a + L::vt_off, 128, L::sbo_vt, kSwzNone);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t s = c % NS, vb = c % NVT, ob = c % NUB;
            PW(0, mbar_wait(&bars[BI.full + s], (c / NS) & 1));
            if (CS > 1 || c >= (uint32_t)NUB) PW(1, mbar_wait(&bars[BI.u_empty + ob], ((c / NUB) & 1) ^ 1));
            PW(2, mbar_wait(&bars[BI.vt_full + vb], (c / NVT) & 1));
            tc_fence_after_sync();
            const uint64_t dK = smem_desc_advance(dK0, s * L::stage_bytes), dV = smem_desc_advance(dV0, vb * L::vt_bytes);
            const uint32_t dU = tb + L::tm_u + ob * 2 * W;
#pragma unroll
            for (int ks = 0; ks < kC / 16; ++ks)
                mma_bf16_ss_w(dU, smem_desc_advance(dK, 2 * ks * 1024), smem_desc_advance(dV, 2 * ks * 128), idU, ks > 0);
            mma_commit_w(&bars[BI.u_done + c % NU]);
            commit_all(&bars[BI.empty + s]);
            if (lane == 0) TC_TRACE(3, c);
        }
    } else if (warp == L::kO2Warp) {
        // ================= issuer: O2 = A_hi V + A_lo V (A operand FROM TMEM, B operand = the V tile, MN-major) =================
        constexpr uint32_t idO2 = idesc_bf16(kC, W, 0, 1);
        constexpr uint32_t sbo_v = 8 * W * 2;     // eight token rows of the V tile
        const uint64_t dV0 = smem_desc(sm_a + L::v_off, 2 * sbo_v, sbo_v, W == 16 ? kSwz32 : kSwz64);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t pb = c % NB, ob = c & 1, vi = c % NV;
            if (CS > 1 || c >= 2) PW(0, mbar_wait(&bars[BI.o2_empty + ob], ((c >> 1) & 1) ^ 1));
            PW(1, mbar_wait(&bars[BI.v_full + vi], (c / NV) & 1));
            PW(2, mbar_wait(&bars[BI.a_full + pb], (c / NB) & 1));
            tc_fence_after_sync();
            if (lane == 0) TC_TRACE(4, c);
            const uint64_t dV = smem_desc_advance(dV0, vi * L::v_bytes);
            const uint32_t dO = tb + L::tm_o2 + ob * W, aA = tb + L::tm_po + pb * NPO;
            // per 16-key step ks the A terms sit where P's columns were: hi pairs at 16 ks .. +8, lo pairs at 16 ks + 8 .. +8
#pragma unroll
            for (int term = 0; term < 2; ++term) {
#pragma unroll
                for (int ks = 0; ks < kC / 16; ++ks)
                    mma_bf16_ts_w(dO, aA + 16 * ks + 8 * term, smem_desc_advance(dV, 2 * ks * sbo_v), idO2, (term | ks) > 0);
            }
            mma_commit_w(&bars[BI.o2_done + vi]);
            if (lane == 0) TC_TRACE(9, c);
        }
    } else if (warp >= 4 && warp < 8) {
        // ================= V~ warps: [V~_hi | V~_lo], V~_j = 2^(b_C - b_j) v_j =================
        // UMMA B operand, MN-major interleaved: (n, k = token) -> (n/8) sbo_vt + (k/8) 128 + (k%8) 16 + (n%8) 2
        const int tid_v = (warp - 4) * 32 + lane;
        constexpr int CG = W / 8;   // 16-byte column groups of a V row
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t vi = c % NV, vb = c % NVT, bt = c / kCPB, gslot = bt & 1;
            if ((c % kCPB) == 0) PW(0, mbar_wait(&bars[BI.g_full + gslot], (bt >> 1) & 1));
            const float* b2 = gate + gslot * 2 * kGateBatch + (c % kCPB) * kC;
            PW(1, mbar_wait(&bars[BI.v_full + vi], (c / NV) & 1));
            // operand buffer vb is free once U(c - NVT) has completed (the U issuer is never ahead of these warps)
            if (c >= (uint32_t)NVT) PW(2, mbar_wait(&bars[BI.u_done + (c - NVT) % NU], ((c - NVT) / NU) & 1));
            const uint8_t* vs = sm + L::v_off + vi * L::v_bytes;
            uint8_t* vt = sm + L::vt_off + vb * L::vt_bytes;
            const float b_last = b2[kC - 1];
#pragma unroll
            for (int it = 0; it < kC * CG / kVtThreads; ++it) {
                const int idx = tid_v + it * kVtThreads, j = idx / CG, cg = idx % CG;
                // undo the TMA swizzle of the V tile: 16-byte chunk index ^= address bits [7, 7 + log2 CG)
                const int sw = (W == 16) ? ((j >> 2) & 1) : ((j >> 1) & 3);
                const uint4 raw = *reinterpret_cast<const uint4*>(vs + j * (W * 2) + ((cg ^ sw) * 16));
                const float sc = ex2(b_last - b2[j]);
                const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
                uint32_t hi[4], lo[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float2 x = fmul2(make_float2(__uint_as_float(w[e] << 16), __uint_as_float(w[e] & 0xFFFF0000u)), make_float2(sc, sc));
                    hi[e] = split2(x.x, x.y, lo[e]);
                }
                const uint32_t off = cg * L::sbo_vt + (j >> 3) * 128 + (j & 7) * 16;
                *reinterpret_cast<uint4*>(vt + off) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                *reinterpret_cast<uint4*>(vt + CG * L::sbo_vt + off) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
            }
            fence_proxy_async_smem();   // generic-proxy writes -> visible to tcgen05.mma's operand reads
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bars[BI.vt_full + vb]);
                mbar_arrive(&bars[BI.v_read + vi]);
                if ((c % kCPB) == (uint32_t)kCPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
            }
        }
    } else if (warp >= 8 && warp < 16) {
        // ================= score warps: A = P (.) 2^(b_i - b_j) (causal), bf16 hi | lo, IN PLACE in TMEM =================
        // A quadrant holds 16 rows of the M = 64 tile (row r in lane 32 (r / 16) + r % 16).  Two warps per quadrant: set 0 takes
        // the key steps 0, 1 (keys 0..31), set 1 the steps 2, 3.  Step ks of quadrant q is all above the diagonal when ks > q
        // (zeros are stored, P is not read), on the diagonal when ks == q (masked), below it otherwise (no mask).
        const int set = (warp - 8) >> 2;
        const int ra = 16 * q + (lane >> 2), rb = ra + 8;
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t pb = c % NB, bt = c / kCPB, gslot = bt & 1;
            if ((c % kCPB) == 0) PW(0, mbar_wait(&bars[BI.g_full + gslot], (bt >> 1) & 1));
            const float* b2 = gate + gslot * 2 * kGateBatch + (c % kCPB) * kC;
            const float bia = b2[ra], bib = b2[rb];
            float2 bj[2][2];
#pragma unroll
            for (int e = 0; e < 2; ++e)
#pragma unroll
                for (int j = 0; j < 2; ++j) bj[e][j] = *reinterpret_cast<const float2*>(b2 + 16 * (2 * set + e) + 8 * j + 2 * (lane & 3));
            PW(1, mbar_wait(&bars[BI.po_full + pb], (c / NB) & 1));
            tc_fence_after_sync();
            if (q == 3 && lane == 0) TC_TRACE(5, c);
            const uint32_t base = tmem_addr(tb, 32 * q, L::tm_po + pb * NPO);
            uint32_t r[2][8];
#pragma unroll
            for (int e = 0; e < 2; ++e)
                if (2 * set + e <= q) tmem_ld_16x256b_x2(base + 16 * (2 * set + e), r[e]);
            PW(2, tmem_ld_wait());
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int ks = 2 * set + e;
                uint32_t hi[4], lo[4];   // {row a block 0, row b block 0, row a block 1, row b block 1}: the 16x128b.x2 fragment
                if (ks <= q) {
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        // (packed fp32: one FADD2 / FMUL2 per pair of columns)
                        const float2 nbj = make_float2(-bj[e][j].x, -bj[e][j].y);
                        const float2 xa = fadd2(make_float2(bia, bia), nbj), xc = fadd2(make_float2(bib, bib), nbj);
                        const float2 pa = fmul2(make_float2(__uint_as_float(r[e][4 * j + 0]), __uint_as_float(r[e][4 * j + 1])), make_float2(ex2(xa.x), ex2(xa.y)));
                        const float2 pc = fmul2(make_float2(__uint_as_float(r[e][4 * j + 2]), __uint_as_float(r[e][4 * j + 3])), make_float2(ex2(xc.x), ex2(xc.y)));
                        float a0 = pa.x, a1 = pa.y, c0 = pc.x, c1 = pc.y;
                        if (ks == q) {   // the diagonal step: causal mask j <= i
                            const int j0 = 16 * ks + 8 * j + 2 * (lane & 3);
                            a0 = (j0 <= ra) ? a0 : 0.f;
                            a1 = (j0 + 1 <= ra) ? a1 : 0.f;
                            c0 = (j0 <= rb) ? c0 : 0.f;
                            c1 = (j0 + 1 <= rb) ? c1 : 0.f;
                        }
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
            PW(3, tmem_st_wait());
            tc_fence_before_sync();
            __syncwarp();
            if (q == 3 && lane == 0) TC_TRACE(6, c);
            if (lane == 0) {
                mbar_arrive(&bars[BI.a_full + pb]);
                if ((c % kCPB) == (uint32_t)kCPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
            }
        }
    } else if (warp >= 16 && warp < 20) {
        // ================= epilogue warps: o_i = 2^(b_i) (O1h_i + O1l_i) + O2_i =================
        // O1(c) is complete with [P|O1](c), long before O2(c): it is read (and its hi + lo terms summed and scaled) as soon as it
        // is there and the accumulator buffer released, so that the buffer's reuse waits for O2's A reads only (r02 timeline: the
        // epilogue's release was the last event of the buffer's life and set the period at W = 32)
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t pb = c % NB, ob = c & 1, bt = c / kCPB, gslot = bt & 1;
            if ((c % kCPB) == 0) PW(0, mbar_wait(&bars[BI.g_full + gslot], (bt >> 1) & 1));
            const float* eb = gate + gslot * 2 * kGateBatch + kGateBatch + (c % kCPB) * kC;
            const int ra = 16 * q + (lane >> 2), rb = ra + 8;
            const float ea = eb[ra], ebb = eb[rb];
            const uint32_t lane_base = 32 * q;
            PW(2, mbar_wait(&bars[BI.po_full + pb], (c / NB) & 1));
            tc_fence_after_sync();
            if (q == 3 && lane == 0) TC_TRACE(10, c);
            float o1[W / 16][8];   // 2^(b_i) (O1h + O1l), fragment layout of the 16x256b loads
#pragma unroll
            for (int cg = 0; cg < W / 16; ++cg) {
                uint32_t r1h[8], r1l[8];
                tmem_ld_16x256b_x2(tmem_addr(tb, lane_base, L::tm_po + pb * NPO + kC + 16 * cg), r1h);
                tmem_ld_16x256b_x2(tmem_addr(tb, lane_base, L::tm_po + pb * NPO + kC + W + 16 * cg), r1l);
                tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 8; i += 2) {
                    const float2 t = fadd2(make_float2(__uint_as_float(r1h[i]), __uint_as_float(r1h[i + 1])), make_float2(__uint_as_float(r1l[i]), __uint_as_float(r1l[i + 1])));
                    o1[cg][i] = t.x;
                    o1[cg][i + 1] = t.y;
                }
            }
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bars[BI.po_read + pb]);
                if ((c % kCPB) == kCPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
            }
            PW(1, mbar_wait(&bars[BI.o2_done + c % NV], (c / NV) & 1));
            tc_fence_after_sync();
            const uint64_t t0 = (uint64_t)c * kC;
            const int n = (int)((T - t0) < (uint64_t)kC ? (T - t0) : (uint64_t)kC);
            OutT* oa = o + (((size_t)b * t_stride + t0 + ra) * H + h) * DV + dv0 + 2 * (lane & 3);
            OutT* oc = o + (((size_t)b * t_stride + t0 + rb) * H + h) * DV + dv0 + 2 * (lane & 3);
            uint32_t r2[W / 16][8];
#pragma unroll
            for (int cg = 0; cg < W / 16; ++cg) tmem_ld_16x256b_x2(tmem_addr(tb, lane_base, L::tm_o2 + ob * W + 16 * cg), r2[cg]);
            tmem_ld_wait();
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BI.o2_empty + ob]);
#pragma unroll
            for (int cg = 0; cg < W / 16; ++cg)
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {   // columns 16 cg + 8 jb + 2 (t % 4) + {0, 1}
                    const float2 va = ffma2(make_float2(ea, ea), make_float2(o1[cg][4 * jb + 0], o1[cg][4 * jb + 1]),
                                            make_float2(__uint_as_float(r2[cg][4 * jb + 0]), __uint_as_float(r2[cg][4 * jb + 1])));
                    const float2 vc = ffma2(make_float2(ebb, ebb), make_float2(o1[cg][4 * jb + 2], o1[cg][4 * jb + 3]),
                                            make_float2(__uint_as_float(r2[cg][4 * jb + 2]), __uint_as_float(r2[cg][4 * jb + 3])));
                    if (ra < n) store_o2<OutT>(oa + 16 * cg + jb * 8, va.x, va.y);
                    if (rb < n) store_o2<OutT>(oc + 16 * cg + jb * 8, vc.x, vc.y);
                }
            if (q == 3 && lane == 0) TC_TRACE(8, c);
        }
    } else if (warp >= 20 && warp < 20 + 4 * NSW) {
        // ================= state warps: the carry  S <- 2^(b_C) S + (Uh + Ul), fp32 FMA in registers =================
        // A warp owns the 32 rows of its TMEM lane quadrant (16 when d_k = 64) x 16 columns of the slice (W = 32: two warps per
        // quadrant), held in the 16x256b fragment layout: per 16-row group lg and 8-column block jb a thread has rows
        // {t/4, t/4 + 8} x columns 2 (t%4) + {0, 1}.  That is the mma fragment layout, so the bf16 hi / lo terms of S go to
        // shared memory TRANSPOSED with stmatrix (.trans): an 8 x 8 block lands as eight 16-byte rows (one column n of S, eight
        // consecutive k) — exactly one swizzle chunk of the K-major [P|O1] operand each.  (The first version of this kernel kept
        // one row per thread and wrote 32 two-byte stores per thread and chunk: the state warps were the busiest role of the
        // CTA, 1080 of 1440 cycles per chunk at W = 16 and 1850 of 2250 at W = 32, r02 wait accounting.)
        constexpr int NLG = (DK == 128) ? 2 : 1;           // 16-row groups per warp
        const int cset = (warp - 20) >> 2;
        const uint32_t col0 = 16 * cset;                   // first column inside the slice
        const uint32_t kq = (DK == 128) ? 32 * q : 16 * q; // first row of the warp
        float S[NLG][2][4];
#pragma unroll
        for (int lg = 0; lg < NLG; ++lg)
#pragma unroll
            for (int jb = 0; jb < 2; ++jb)
#pragma unroll
                for (int hl = 0; hl < 2; ++hl) {
                    float2 x = make_float2(0.f, 0.f);
                    if (state_in)
                        x = *reinterpret_cast<const float2*>(state_in + ((size_t)bh * DK + kq + 16 * lg + 8 * hl + (lane >> 2)) * DV + dv0 + col0 +
                                                             8 * jb + 2 * (lane & 3));
                    S[lg][jb][2 * hl] = x.x;
                    S[lg][jb][2 * hl + 1] = x.y;
                }
        // stmatrix row addresses: lane L supplies row L % 8 (column n of S) of matrix L / 8 = {hi rows 0-7, hi rows 8-15, lo rows 0-7,
        // lo rows 8-15} of the (lg, jb) block; operand row R = 64 + term W + col0 + 8 jb + n, chunk ((k0 % 64) / 8) ^ (R % 8)
        uint32_t st_off[NLG][2];
#pragma unroll
        for (int lg = 0; lg < NLG; ++lg)
#pragma unroll
            for (int jb = 0; jb < 2; ++jb) {
                const uint32_t term = lane >> 4, hl = (lane >> 3) & 1, n = lane & 7;
                const uint32_t R = kC + term * W + col0 + 8 * jb + n, k0 = kq + 16 * lg + 8 * hl;
                st_off[lg][jb] = L::q_bytes + (k0 >> 6) * L::ks_half_bytes + R * 128 + ((((k0 & 63) >> 3) ^ (R & 7)) << 4);
            }
        auto write_s_operand = [&](uint32_t s) {
            const uint32_t stage = sm_a + L::stage_off + s * L::stage_bytes;
#pragma unroll
            for (int lg = 0; lg < NLG; ++lg)
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {
                    uint32_t lo0, lo1;
                    const uint32_t hi0 = split2(S[lg][jb][0], S[lg][jb][1], lo0), hi1 = split2(S[lg][jb][2], S[lg][jb][3], lo1);
                    stmatrix_x4_trans(stage + st_off[lg][jb], hi0, hi1, lo0, lo1);
                }
        };
        write_s_operand(0);   // version 0 of the S operand (read by [P|O1](0)); stage 0 is fresh
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars[BI.s_full]);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t ob = c % NUB, bt = c / kCPB, gslot = bt & 1;
            if ((c % kCPB) == 0) PW(0, mbar_wait(&bars[BI.g_full + gslot], (bt >> 1) & 1));
            const float gam = gate[gslot * 2 * kGateBatch + kGateBatch + (c % kCPB) * kC + kC - 1];
            PW(1, mbar_wait(&bars[BI.u_done + c % NU], (c / NU) & 1));
            tc_fence_after_sync();
            if (q == 3 && lane == 0) TC_TRACE(2, c);
            uint32_t uh[NLG][8], ul[NLG][8];
#pragma unroll
            for (int lg = 0; lg < NLG; ++lg) {
                tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q + 16 * lg, L::tm_u + ob * 2 * W + col0), uh[lg]);
                tmem_ld_16x256b_x2(tmem_addr(tb, 32 * q + 16 * lg, L::tm_u + ob * 2 * W + W + col0), ul[lg]);
            }
            tmem_ld_wait();
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bars[BI.u_empty + ob]);
                if ((c % kCPB) == kCPB - 1 || c + 1 == n_chunks) mbar_arrive(&bars[BI.g_empty + gslot]);
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
            if (c + 1 < n_chunks) {   // version c+1 of the S operand, into the stage chunk c+1 lands in
                const uint32_t s1 = (c + 1) % NS;
                if (CS > 1 || c + 1 >= (uint32_t)NS) PW(2, mbar_wait(&bars[BI.empty + s1], ((((c + 1) / NS) & 1) ^ 1)));   // chunk c+1-NS is done with that stage
                write_s_operand(s1);
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars[BI.s_full + s1]);
            }
            if (q == 3 && lane == 0) TC_TRACE(7, c);
        }
#pragma unroll
        for (int lg = 0; lg < NLG; ++lg)
#pragma unroll
            for (int jb = 0; jb < 2; ++jb)
#pragma unroll
                for (int hl = 0; hl < 2; ++hl)
                    *reinterpret_cast<float2*>(state_out + ((size_t)bh * DK + kq + 16 * lg + 8 * hl + (lane >> 2)) * DV + dv0 + col0 + 8 * jb +
                                               2 * (lane & 3)) = make_float2(S[lg][jb][2 * hl], S[lg][jb][2 * hl + 1]);
    }

    PROF_END;
    if (threadIdx.x == 0) TC_TRACE(13, 0);
    // ---- teardown: every tcgen05 op of this CTA has completed (the state and epilogue warps waited on the last commits),
    // and no peer still multicasts or arrives into this CTA once the whole cluster is here ----
    tc_fence_before_sync();
    if constexpr (CS > 1) cluster_sync_relaxed();
    else __syncthreads();
    if (warp == 2) tmem_dealloc(tb, L::tmem_cols);
    if (threadIdx.x == 0) TC_TRACE(15, 0);
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
int make_tmap(CUtensorMap* m, const void* base, uint32_t D, uint32_t H, uint64_t T, uint64_t t_stride, uint32_t B,
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

// whole Q tiles for the cluster-free launch: dimensions (d % 64, t, d / 64, h, b), box (64, box_t, D / 64, 1, 1)
int make_tmap_halves(CUtensorMap* m, const void* base, uint32_t D, uint32_t H, uint64_t T, uint64_t t_stride, uint32_t B,
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

template <int DK, int W, int CS, typename OutT>
static int launch_scan_t(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g,
                         const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    using L = ScanCfg<DK, W, CS>;
    // one attribute slot per instantiation: DK (2) x W (2) x CS (3) x OutT (2)
    constexpr uint32_t slot = kSlotScan + (DK == 128 ? 0 : 1) + 2 * (W == 16 ? 0 : 1) + 4 * (CS == 1 ? 0 : (CS == 2 ? 1 : 2)) +
                              12 * (sizeof(OutT) == 4 ? 0 : 1);
    {
        const int rc = ensure_dyn_smem(ctx, slot, esc_scan_kernel<DK, W, CS, OutT>, (int)L::total);
        if (rc != ESC_OK) return rc;
    }
    if (!state_out) return ESC_OK;   // prepare-only call (before a stream capture)
    CUtensorMap tq, tk, tv, tqp, tkp;   // tqp / tkp: whole [64 x d_k] tiles through the 5-D halves map (L2 prefetches; Q loads without a cluster)
    const void* qq = T ? q : (const void*)state_out;   // T == 0: maps are never dereferenced, any valid address will do
    const void* kk = T ? k : (const void*)state_out;
    const void* vv = T ? v : (const void*)state_out;
    const uint64_t ts = t_stride ? t_stride : 1;
    // Q / K: each CTA of the cluster loads (and multicasts) 64 / CS rows of a chunk; V: the CTA's own W columns
    int rc = make_tmap_halves(&tqp, qq, DK, s.H, T, ts, s.B, kC);
    if (rc == ESC_OK) rc = make_tmap_halves(&tkp, kk, DK, s.H, T, ts, s.B, kC);
    if (rc != ESC_OK) return rc;
    if (CS == 1) tq = tqp;
    else rc = make_tmap(&tq, qq, DK, s.H, T, ts, s.B, 64, kC / CS, CU_TENSOR_MAP_SWIZZLE_128B);
    if (rc == ESC_OK) rc = make_tmap(&tk, kk, DK, s.H, T, ts, s.B, 64, kC / CS, CU_TENSOR_MAP_SWIZZLE_128B);
    if (rc == ESC_OK) rc = make_tmap(&tv, vv, s.dv, s.H, T, ts, s.B, W, kC, W == 16 ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_64B);
    if (rc != ESC_OK) return rc;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(s.dv / W, s.B * s.H);   // d_v / W CTAs per (b, h), in clusters of CS
    cfg.blockDim = dim3(L::kThreads);
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
    ESC_CUDA(cudaLaunchKernelEx(&cfg, esc_scan_kernel<DK, W, CS, OutT>, tq, tk, tv, tqp, tkp, g, state_in, state_out, (OutT*)o, s.H, s.dv, T,
                                t_stride));
    return ESC_OK;
}

template <int DK, int W, int CS>
static int launch_scan_o(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g,
                         const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    if (s.out_dtype == ESC_DTYPE_F32) return launch_scan_t<DK, W, CS, float>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    return launch_scan_t<DK, W, CS, bf16>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
}

// d_v columns per CTA: a function of the shape key ONLY (never of T).  16 columns while that still fits the device in one
// wave of one-CTA-per-SM blocks (B H d_v / 16 <= SMs: B = 1 of the paper-shaped workloads), else 32: at 16 columns the fixed
// per-chunk cost of a CTA (Q, K through shared memory, the scores) is paid for half as many outputs, which only pays off
// when it buys SMs that would otherwise idle.
uint32_t scan_tile_columns(const esc_ctx* ctx, const ScanShape& s) {
    const uint64_t ctas16 = (uint64_t)s.B * s.H * (s.dv / 16);
    const uint64_t sms = ctx && ctx->sm_count > 0 ? (uint64_t)ctx->sm_count : 148u;
    return (ctas16 > sms && s.dv % 32 == 0) ? 32u : 16u;
}

// Calls of up to kShortT tokens (the suffix scan after a restore: one or two chunks) launch WITHOUT the cluster: whole-tile
// TMA loads instead of multicast row slices, no cluster barrier at set-up and teardown.  A one-chunk call is a single pass
// through the dependent pipeline, and the cluster's benefit (L2 -> SM traffic of Q / K divided by the cluster size) only
// shows over many chunks.  The MMAs, their operands and their order are the same: the launches are bit-identical.
#ifndef ESC_SCAN_SHORT
#define ESC_SCAN_SHORT 128
#endif
constexpr uint64_t kShortT = ESC_SCAN_SHORT;

template <int DK, int W>
static int launch_scan_w(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g,
                         const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    const uint32_t per_head = s.dv / W;                 // CTAs per (b, h)
    const bool pair = per_head % 4 != 0;                // d_v = 64 with 32-column tiles: clusters of two
    if (per_head % 2 != 0) return ESC_ERR_UNSUPPORTED;
    if (!state_out) {   // prepare-only call: both launch forms
        const int rc = launch_scan_o<DK, W, 1>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
        if (rc != ESC_OK) return rc;
    } else if (T <= kShortT) {
        return launch_scan_o<DK, W, 1>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    }
    if constexpr (W == 32) {
        if (pair) return launch_scan_o<DK, W, 2>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    }
    return launch_scan_o<DK, W, 4>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
}

// The key's chunk (64 or 128) is the alignment grid the caller commits to (restore boundaries are multiples of it); the
// kernel's token tile is 64 for both: the recurrence is the same function, and a 128-aligned boundary is also 64-aligned
// (so restore + continue stays bit-identical to the cold run).
int launch_scan_tc(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g,
                   const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    if (s.chunk != 64 && s.chunk != 128) return ESC_ERR_UNSUPPORTED;
    const uint32_t w = scan_tile_columns(ctx, s);
    if (s.dk == 128) {
        if (w == 32) return launch_scan_w<128, 32>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
        return launch_scan_w<128, 16>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    }
    if (s.dk == 64) {
        if (w == 32) return launch_scan_w<64, 32>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
        return launch_scan_w<64, 16>(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
    }
    return ESC_ERR_UNSUPPORTED;
}

#ifdef ESC_SCAN_PROF
extern "C" int esc_debug_scan_prof_read(long long* host) {
    return (int)cudaMemcpyFromSymbol(host, g_scan_prof, sizeof(g_scan_prof));
}
#endif
#ifdef ESC_TC_TRACE
extern "C" int esc_debug_trace_read(long long* host) {
    return (int)cudaMemcpyFromSymbol(host, g_tc_trace, sizeof(g_tc_trace));
}
#endif

}  // namespace esc
