// Internal structures of libesc (host side) + the device copy-table layout.
// The public contract is include/esc.h; nothing here crosses the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <atomic>
#include <memory>
#include <string>
#include <utility>
#include <vector>

#include "esc.h"

namespace esc {

// ---- error plumbing -------------------------------------------------------------------
extern thread_local int g_last_cuda_error;
inline int cuda_fail(cudaError_t e) {
    g_last_cuda_error = (int)e;
    return ESC_ERR_CUDA;
}
#define ESC_CUDA(call)                                        \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return ::esc::cuda_fail(e__); \
    } while (0)

// ---- copy table (what the capsule copy kernel consumes) --------------------------------
// One entry per (row, segment): `bytes` valid bytes from src to dst[0..n_dst).
// Tiles of kCopyTileBytes are numbered globally; tile_begin[i] is the first tile of entry i.
constexpr uint32_t kCopyThreads = 256;
constexpr uint32_t kCopyUnroll = 2;                    // 16-byte vectors in flight per thread
constexpr uint32_t kCopyTileBytes = kCopyThreads * kCopyUnroll * 16u;   // 8 KiB
constexpr uint32_t kCopyMaxSeg = 112;                 // entries per launch (table <= 4 KiB kernel params)
constexpr uint32_t kCopyMaxSegFork = 96;              // entries per fork launch

struct CopyTable {                                    // single destination: 3600 B
    uint32_t n_seg;
    uint32_t n_tiles;
    uint32_t tile_begin[kCopyMaxSeg + 1];
    uint32_t pad_;
    const uint8_t* src[kCopyMaxSeg];
    uint8_t* dst[kCopyMaxSeg];
    uint64_t bytes[kCopyMaxSeg];
};

struct ForkTable {                                    // n_dst destinations (large kernel params)
    uint32_t n_seg;
    uint32_t n_tiles;
    uint32_t n_dst;
    uint32_t pad_;
    uint32_t tile_begin[kCopyMaxSegFork + 1];
    uint32_t pad2_;
    const uint8_t* src[kCopyMaxSegFork];
    uint64_t bytes[kCopyMaxSegFork];
    uint8_t* dst[ESC_MAX_FORK][kCopyMaxSegFork];
};

// ---- handles ----------------------------------------------------------------------------
struct Row {                          // plain data: copying a row table allocates nothing (names live in esc_bufset::names)
    uint8_t* base;
    uint64_t capacity, fixed_bytes, bytes_per_token, seg_stride;
    uint32_t n_seg;
    // optional BF16 dequantisation stage of an FP8 row (include/esc.h "FP8 KV rows"); not part of the capsule
    uint8_t* stage = nullptr;
    uint32_t stage_format = 0;
    float stage_scale = 1.f;
    uint64_t stage_valid_tokens = 0;
};

}  // namespace esc

struct esc_graph;
struct esc_ctx {
    int device;
    int sm_count;
    int l2_bytes;
    // kernel instantiations whose max-dynamic-shared-memory attribute has been set on THIS context's device (the attribute
    // is per device; a process-wide flag would leave a second context's device at the 48 KiB default)
    std::atomic<uint64_t> func_attr_mask{0};
    // Graph[key] table (include/esc.h): most recently used first
    std::vector<std::pair<uint64_t, esc_graph*>> plans;
    uint32_t plan_capacity = 8;
    uint64_t plan_hits = 0, plan_misses = 0, plan_evictions = 0;
};

namespace esc {
struct Seg {                          // host-side flattened (row, segment) of a live<->slab pairing
    uint8_t* live;
    uint64_t slab_off;
    uint64_t bytes;
};
struct SegCache {                     // the flattened segment table of a live set at one boundary (hot path: no rebuild per verb)
    bool valid = false;
    uint64_t P = 0, slab_bytes = 0, payload_bytes = 0;
    std::vector<Seg> segs;
};
}  // namespace esc

struct esc_bufset {
    esc_ctx* ctx;
    bool frozen;                      // false: live set; true: capsule
    std::vector<esc::Row> rows;       // live: the registered buffers.  capsule: layout copy (base = nullptr)
    std::shared_ptr<const std::vector<std::string>> names;   // row names, shared between a live set and its capsules
    esc::SegCache seg_cache;          // live sets: last boundary walked (snapshot / restore / fork / set_capsule)
    uint64_t layout_digest;
    uint64_t position;                // live: current token position; capsule: boundary P'
    // capsule only
    uint8_t* slab;                    // device address the copy kernels read (HOST tier: the pinned slab's device alias)
    uint8_t* slab_host;               // HOST tier: the pinned host address; GPU tier: nullptr
    uint32_t tier;                    // ESC_TIER_GPU / ESC_TIER_HOST
    uint64_t slab_bytes, payload_bytes, chunk, prefix_digest;
};

namespace esc {

// Every verb runs on its context's device whatever the caller's current device is, and leaves the caller's current
// device as it found it (include/esc.h "Devices").
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(const esc_ctx* c) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != c->device) {
            err = cudaSetDevice(c->device);
            switched = err == cudaSuccess;
        }
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define ESC_ON_DEVICE(ctx)                 \
    ::esc::DeviceGuard dev_guard__(ctx);   \
    if (dev_guard__.err != cudaSuccess) return ::esc::cuda_fail(dev_guard__.err)

// cudaFuncAttributeMaxDynamicSharedMemorySize, once per (context, kernel instantiation `slot`); idempotent, so two threads
// racing on the same slot only set it twice
enum FuncSlot : uint32_t { kSlotGdn = 0, kSlotScan = 4 };   // scan instantiations take kSlotScan + their own index
template <typename K>
int ensure_dyn_smem(esc_ctx* ctx, uint32_t slot, K kernel, int bytes) {
    const uint64_t bit = 1ull << slot;
    if (ctx->func_attr_mask.load(std::memory_order_acquire) & bit) return ESC_OK;
    ESC_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    ctx->func_attr_mask.fetch_or(bit, std::memory_order_release);
    return ESC_OK;
}

uint64_t seg_valid(const Row& r, uint64_t P);
int check_fit(const std::vector<Row>& rows, uint64_t P);
// slab layout walk: fills segs (live pointers relative to `rows`), returns slab bytes / payload
void layout_walk(const std::vector<Row>& rows, uint64_t P, std::vector<Seg>* segs, uint64_t* slab_bytes,
                 uint64_t* payload_bytes);
// the same walk through the live set's one-entry cache (rebuilt only when P changes)
const SegCache& live_segs(esc_bufset* live, uint64_t P);
// one copy-kernel launch per kCopyMaxSeg segments: live -> slab (to_slab) or slab -> live
int launch_copy_segs(const esc_ctx* ctx, const std::vector<Seg>& segs, uint8_t* slab, bool to_slab, cudaStream_t stream);
// the restore node's table for (live segments, capsule slab)
void build_restore_table(CopyTable* t, const std::vector<Seg>& segs, const uint8_t* slab);

// copy kernel launchers (copy_kernel.cu)
uint32_t copy_grid_blocks(uint64_t n_tiles);
// Launch the copy of `n` (src,dst,bytes) entries, splitting into several launches only when n > kCopyMaxSeg.
int launch_copy(const esc_ctx* ctx, const uint8_t* const* src, uint8_t* const* dst, const uint64_t* bytes, uint32_t n,
                cudaStream_t stream);
int launch_fork(const esc_ctx* ctx, const uint8_t* const* src, uint8_t* const* const* dst, uint32_t n_dst,
                const uint64_t* bytes, uint32_t n, cudaStream_t stream);
// table-in-global-memory variant used inside captured graphs
void build_copy_table(CopyTable* t, const uint8_t* const* src, uint8_t* const* dst, const uint64_t* bytes, uint32_t n);
int launch_copy_indirect(const esc_ctx* ctx, const CopyTable* table_dev, uint32_t grid_blocks, cudaStream_t stream);
// stores t (passed by value as a kernel parameter) to the device-resident table on `stream`
int launch_table_store(const CopyTable& t, CopyTable* table_dev, cudaStream_t stream);

// staged copy / FP8 -> BF16 expansion (stage.cu): entry i copies bytes[i] from src to dst8 (if not NULL) and writes
// their BF16 expansion to dst16 (if not NULL)
int launch_stage(const esc_ctx* ctx, const uint8_t* const* src, uint8_t* const* dst8, uint8_t* const* dst16,
                 const uint64_t* bytes, const float* scale, uint32_t n, cudaStream_t stream);
void reset_stage_valid(esc_bufset* live, uint64_t tokens);

// scan (scan_kernel.cu)
struct ScanShape {
    uint32_t B, H, dk, dv, in_dtype, out_dtype, chunk;
};
bool decode_key(esc_shape_key key, ScanShape* s);
// d_v columns per CTA of the scan kernel: a function of the shape key (and the device's SM count) only, never of T
uint32_t scan_tile_columns(const esc_ctx* ctx, const ScanShape& s);
int launch_scan(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g,
                const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream);
// gated delta rule, chunked (WY) form on tcgen05 (gdn_scan_kernel.cu)
int launch_gdn_mma(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* beta,
                   const float* state_in, float* state_out, float* o, uint64_t T, uint64_t t_stride, cudaStream_t stream);

}  // namespace esc
