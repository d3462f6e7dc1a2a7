// Capsule copy kernel: one launch moves every (row, segment) of a named buffer set.
//
// PAPER.md:117-132 (Algorithm 1) makes snapshot / restore / fork / rollback "a single copy of
// that buffer set" — Θ(bytes), bandwidth-bound (Table 3).  The paper
// does not say how its device-to-device copy is issued; here it is ONE kernel driven by a
// descriptor table (kernel parameter space, or a device-resident table inside captured
// graphs), so a 24-30 buffer capsule pays one launch, not 30 memcpy nodes.
//
// Roofline: HBM.  Algorithmic bytes = 2 x capsule bytes (read + write), (1 + n) x for an n-way
// fork.  Work decomposition: the byte ranges are cut into tiles of kCopyTileBytes (8 KiB)
// numbered globally, ONE CTA PER TILE (the grid is the tile count: 8 448 CTAs for the 66 MiB
// capsule, 51 456 at 402 MiB), so the hardware block scheduler balances the SMs and the tail.
// Measured on B200 (r01 sweep, clean L2, CUDA events): a persistent grid of 148 x 8 CTAs striding
// over 16 KiB tiles reached 6.0 TB/s at 402 MiB, one CTA per 8 KiB tile 6.8 TB/s.  A tile is
// moved with 16-byte vector loads/stores (L1 no-allocate), all loads of a thread issued before
// its first store; 8 resident CTAs x 256 threads x 2 x 16 B = 64 KiB in flight per SM.
// Odd tails and unaligned pointers take a byte path.
#include <string.h>

#include "esc_internal.h"

namespace esc {

constexpr int kCopyBlocksPerSM = 8;

__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream(uint4* p, const uint4& v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
                 "r"(v.w)
                 : "memory");
}

// entry index of a global tile number: largest i with tile_begin[i] <= tile (zero-tile entries skipped)
__device__ __forceinline__ uint32_t find_entry(const uint32_t* tile_begin, uint32_t n_seg, uint32_t tile) {
    uint32_t lo = 0, hi = n_seg;  // invariant: tile_begin[lo] <= tile < tile_begin[hi]
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (tile_begin[mid] <= tile) lo = mid;
        else hi = mid;
    }
    return lo;
}

template <int kDst>
__device__ __forceinline__ void copy_tile(const uint8_t* __restrict__ src, uint8_t* const* dst, uint32_t n_dst,
                                          uint64_t n) {
    const uint32_t tid = threadIdx.x;
    bool aligned = (((uintptr_t)src) & 15u) == 0;
#pragma unroll
    for (int d = 0; d < kDst; ++d)
        if (d < (int)n_dst) aligned = aligned && ((((uintptr_t)dst[d]) & 15u) == 0);
    if (aligned) {
        const uint4* s = (const uint4*)src;
        if (n == kCopyTileBytes) {  // full tile: all loads first, then all stores
            uint4 v[kCopyUnroll];
#pragma unroll
            for (int u = 0; u < (int)kCopyUnroll; ++u) v[u] = ld_stream(s + tid + u * kCopyThreads);
#pragma unroll
            for (int d = 0; d < kDst; ++d) {
                if (d < (int)n_dst) {
                    uint4* o = (uint4*)dst[d];
#pragma unroll
                    for (int u = 0; u < (int)kCopyUnroll; ++u) st_stream(o + tid + u * kCopyThreads, v[u]);
                }
            }
            return;
        }
        const uint32_t n16 = (uint32_t)(n >> 4);
        for (uint32_t i = tid; i < n16; i += kCopyThreads) {
            const uint4 v = ld_stream(s + i);
#pragma unroll
            for (int d = 0; d < kDst; ++d)
                if (d < (int)n_dst) st_stream((uint4*)dst[d] + i, v);
        }
        for (uint32_t i = (n16 << 4) + tid; i < n; i += kCopyThreads) {
            const uint8_t b = src[i];
#pragma unroll
            for (int d = 0; d < kDst; ++d)
                if (d < (int)n_dst) dst[d][i] = b;
        }
        return;
    }
    for (uint32_t i = tid; i < n; i += kCopyThreads) {  // byte path: exact for any alignment
        const uint8_t b = src[i];
#pragma unroll
        for (int d = 0; d < kDst; ++d)
            if (d < (int)n_dst) dst[d][i] = b;
    }
}

// Programmatic dependent launch (both directions): a copy kernel may be placed while its predecessor on the stream drains
// (nothing is read or written before griddepcontrol.wait), and it lets its successor be placed while its own last wave drains
// (launch_dependents once this CTA's loads are in flight; the successor's own wait still orders it after ALL of this grid's
// stores).  Back-to-back verbs and the restore -> first suffix scan hand-over lose the launch gap (r02).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <bool kWaitFirst>
__device__ __forceinline__ void copy_body(const CopyTable& t) {
    // kWaitFirst: the table itself is in global memory (graph restore node) and may only be read after the dependency wait;
    // a table in kernel-parameter space is searched BEFORE the wait, so that the loads go out the moment the wait returns
    if (kWaitFirst) pdl_wait();
    const uint32_t n_tiles = t.n_tiles, n_seg = t.n_seg;
    bool waited = kWaitFirst;
    for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const uint32_t e = find_entry(t.tile_begin, n_seg, tile);
        const uint64_t off = (uint64_t)(tile - t.tile_begin[e]) * kCopyTileBytes;
        const uint64_t left = t.bytes[e] - off;
        uint8_t* d = t.dst[e] + off;
        const uint8_t* sp = t.src[e] + off;
        if (!waited) {
            pdl_wait();
            waited = true;
        }
        copy_tile<1>(sp, &d, 1, left < kCopyTileBytes ? left : kCopyTileBytes);
    }
    if (!waited) pdl_wait();
    pdl_launch_dependents();
}

// table in kernel-parameter space: no H2D copy, no device allocation per verb
__global__ void __launch_bounds__(kCopyThreads, kCopyBlocksPerSM) esc_copy_kernel(const __grid_constant__ CopyTable t) {
    copy_body<false>(t);
}

// table in global memory: the restore node of a captured graph (PAPER.md:110,128 — the host
// overwrites the bound table between replays; the graph is never recaptured)
__global__ void __launch_bounds__(kCopyThreads, kCopyBlocksPerSM) esc_copy_indirect_kernel(const CopyTable* __restrict__ tp) {
    copy_body<true>(*tp);
}

// fork: read each tile once, write it to n_dst live sets
__global__ void __launch_bounds__(kCopyThreads, kCopyBlocksPerSM) esc_fork_kernel(const __grid_constant__ ForkTable t) {
    pdl_wait();
    const uint32_t n_tiles = t.n_tiles, n_seg = t.n_seg, n_dst = t.n_dst;
    for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const uint32_t e = find_entry(t.tile_begin, n_seg, tile);
        const uint64_t off = (uint64_t)(tile - t.tile_begin[e]) * kCopyTileBytes;
        const uint64_t left = t.bytes[e] - off;
        uint8_t* d[ESC_MAX_FORK];
#pragma unroll
        for (int i = 0; i < (int)ESC_MAX_FORK; ++i) d[i] = i < (int)n_dst ? t.dst[i][e] + off : nullptr;
        copy_tile<ESC_MAX_FORK>(t.src[e] + off, d, n_dst, left < kCopyTileBytes ? left : kCopyTileBytes);
    }
    pdl_launch_dependents();
}

// ---- host -----------------------------------------------------------------------------------
// one CTA per tile; the kernels' grid-stride loop only matters beyond the grid-size limit
uint32_t copy_grid_blocks(uint64_t n_tiles) { return n_tiles < 0x7FFFFFFFull ? (n_tiles ? (uint32_t)n_tiles : 1u) : 0x7FFFFFFFu; }

template <typename K, typename... Args>
static cudaError_t launch_pdl(K kernel, uint32_t grid, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kCopyThreads);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    memset(attr, 0, sizeof attr);
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}

static uint32_t fill_tiles(uint32_t* tile_begin, const uint64_t* bytes, uint32_t n) {
    uint64_t t = 0;
    for (uint32_t i = 0; i < n; ++i) {
        tile_begin[i] = (uint32_t)t;
        t += (bytes[i] + kCopyTileBytes - 1) / kCopyTileBytes;
    }
    tile_begin[n] = (uint32_t)t;
    return (uint32_t)t;
}

void build_copy_table(CopyTable* t, const uint8_t* const* src, uint8_t* const* dst, const uint64_t* bytes, uint32_t n) {
    memset(t, 0, sizeof *t);
    t->n_seg = n;
    t->n_tiles = fill_tiles(t->tile_begin, bytes, n);
    for (uint32_t i = 0; i < n; ++i) {
        t->src[i] = src[i];
        t->dst[i] = dst[i];
        t->bytes[i] = bytes[i];
    }
}

int launch_copy(const esc_ctx* ctx, const uint8_t* const* src, uint8_t* const* dst, const uint64_t* bytes, uint32_t n,
                cudaStream_t stream) {
    for (uint32_t first = 0; first < n; first += kCopyMaxSeg) {
        const uint32_t m = n - first < kCopyMaxSeg ? n - first : kCopyMaxSeg;
        CopyTable t;
        build_copy_table(&t, src + first, dst + first, bytes + first, m);
        if (t.n_tiles == 0) continue;
        (void)ctx;
        ESC_CUDA(launch_pdl(esc_copy_kernel, copy_grid_blocks(t.n_tiles), stream, t));
    }
    return ESC_OK;
}

// Rebinding a captured graph's restore node to another capsule (esc_graph_set_capsule): the new table travels as a kernel
// parameter and one small CTA stores it to the device-resident copy.  No copy engine and no pinned mirror are involved:
// a cudaMemcpyAsync of the table queues behind the caller's own host-to-device transfers on the same engine and needs a
// host-side wait before the mirror can be reused (r01u: 0.42 -> 0.33 ms per end-to-end step, bench.py e2e).
__global__ void __launch_bounds__(kCopyThreads) esc_table_store_kernel(const __grid_constant__ CopyTable t, CopyTable* dst) {
    static_assert(sizeof(CopyTable) % 4 == 0, "word copy");
    const uint32_t* s = reinterpret_cast<const uint32_t*>(&t);
    uint32_t* d = reinterpret_cast<uint32_t*>(dst);
    pdl_wait();   // a replay that still reads the previous table has completed
    for (uint32_t i = threadIdx.x; i < sizeof(CopyTable) / 4; i += kCopyThreads) d[i] = s[i];
    pdl_launch_dependents();
}

int launch_table_store(const CopyTable& t, CopyTable* table_dev, cudaStream_t stream) {
    ESC_CUDA(launch_pdl(esc_table_store_kernel, 1, stream, t, table_dev));
    return ESC_OK;
}

int launch_copy_indirect(const esc_ctx* ctx, const CopyTable* table_dev, uint32_t grid_blocks, cudaStream_t stream) {
    (void)ctx;
    ESC_CUDA(launch_pdl(esc_copy_indirect_kernel, grid_blocks, stream, table_dev));
    return ESC_OK;
}

int launch_fork(const esc_ctx* ctx, const uint8_t* const* src, uint8_t* const* const* dst, uint32_t n_dst,
                const uint64_t* bytes, uint32_t n, cudaStream_t stream) {
    for (uint32_t first = 0; first < n; first += kCopyMaxSegFork) {
        const uint32_t m = n - first < kCopyMaxSegFork ? n - first : kCopyMaxSegFork;
        ForkTable t;
        memset(&t, 0, sizeof t);
        t.n_seg = m;
        t.n_dst = n_dst;
        t.n_tiles = fill_tiles(t.tile_begin, bytes + first, m);
        for (uint32_t i = 0; i < m; ++i) {
            t.src[i] = src[first + i];
            t.bytes[i] = bytes[first + i];
            for (uint32_t d = 0; d < n_dst; ++d) t.dst[d][i] = dst[d][first + i];
        }
        if (t.n_tiles == 0) continue;
        (void)ctx;
        ESC_CUDA(launch_pdl(esc_fork_kernel, copy_grid_blocks(t.n_tiles), stream, t));
    }
    return ESC_OK;
}

}  // namespace esc
