// esc_restore_static (include/esc.h): restore(cap) for callers that cannot provide or allocate scratch memory.
//
// The restore node of a captured graph reads its descriptor table from caller-owned device scratch (graph.cu:
// esc_graph_scratch_bytes / esc_copy_indirect_kernel).  Code that runs under somebody else's stream capture, a tight
// serving loop or a harness that forbids cudaMalloc has no such scratch to hand over.  This entry point drives the SAME
// table-in-global-memory copy kernel, with the table in a file-scope __device__ array of a fixed, modest size that every
// GPU which loads the library holds until exit: kStaticTables tables of kCopyMaxSeg segments each, 13 KiB.  It allocates
// nothing on the device: no cudaMalloc / cudaFree / allocating library routine, two kernel launches per table (the
// one-CTA table store, then the copy).
//
// The array is shared by every call on a device and keeps the last call's tables.  Nothing in it has to start at zero:
// a call overwrites every word of each table it uses before the copy kernel reads it, and never reads a table it did not
// write.  Calls are ordered by the stream they are enqueued on (the table store waits for the preceding kernel of the stream
// under programmatic dependent launch, like esc_graph_set_capsule); two calls whose kernels can overlap on the GPU (different
// streams without an event between them, or different host threads) RACE on the tables: the caller serialises them.
#include <mutex>

#include "esc_internal.h"

namespace esc {

constexpr uint32_t kStaticTables = ESC_RESTORE_STATIC_MAX_SEGMENTS / kCopyMaxSeg;
static_assert(kStaticTables * kCopyMaxSeg == ESC_RESTORE_STATIC_MAX_SEGMENTS, "the public limit is a whole number of tables");
constexpr size_t kStaticTableStride = (sizeof(CopyTable) + 255) / 256 * 256;

// In host code this name is a host-side stand-in for the symbol, NOT a device address: the address the kernels get comes
// from cudaGetSymbolAddress below, once per device.
static __device__ __align__(256) unsigned char g_restore_tables[kStaticTables * kStaticTableStride];

constexpr int kMaxDevices = 64;
static std::mutex g_addr_mu;
static unsigned char* g_addr[kMaxDevices];   // per device ordinal: the array's address on that device (nullptr: not looked up yet)

// the device of `ctx` is current (ESC_ON_DEVICE in the caller)
static int static_tables_on_device(const esc_ctx* ctx, unsigned char** out) {
    if (ctx->device < 0 || ctx->device >= kMaxDevices) return ESC_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_addr_mu);
    if (!g_addr[ctx->device]) {
        void* p = nullptr;
        ESC_CUDA(cudaGetSymbolAddress(&p, g_restore_tables));
        if (!p || ((uintptr_t)p & 255u)) return ESC_ERR_CUDA;
        g_addr[ctx->device] = static_cast<unsigned char*>(p);
    }
    *out = g_addr[ctx->device];
    return ESC_OK;
}

}  // namespace esc

using namespace esc;

extern "C" {

uint32_t esc_restore_static_max_segments(void) { return ESC_RESTORE_STATIC_MAX_SEGMENTS; }

int esc_restore_static(esc_bufset* live, const esc_bufset* capsule, const uint64_t* expect_prefix_digest, void* stream) {
    // the pairing rules of esc_restore
    if (!live || !capsule || live->frozen || !capsule->frozen) return ESC_ERR_INVALID;
    if (live->layout_digest != capsule->layout_digest || live->rows.size() != capsule->rows.size()) return ESC_ERR_MISMATCH;
    int rc = check_fit(live->rows, capsule->position);
    if (rc != ESC_OK) return rc;
    if (expect_prefix_digest && *expect_prefix_digest != capsule->prefix_digest) return ESC_ERR_MISMATCH;
    ESC_ON_DEVICE(live->ctx);
    const std::vector<Seg>& segs = live_segs(live, capsule->position).segs;
    if (segs.size() > ESC_RESTORE_STATIC_MAX_SEGMENTS) return ESC_ERR_CAPACITY;   // more segments than the static tables hold
    unsigned char* base = nullptr;
    rc = static_tables_on_device(live->ctx, &base);
    if (rc != ESC_OK) return rc;
    uint32_t slot = 0;
    for (size_t first = 0; first < segs.size(); first += kCopyMaxSeg, ++slot) {
        const size_t m = segs.size() - first < kCopyMaxSeg ? segs.size() - first : kCopyMaxSeg;
        const std::vector<Seg> part(segs.begin() + first, segs.begin() + first + m);
        CopyTable t;
        build_restore_table(&t, part, capsule->slab);
        if (t.n_tiles == 0) continue;
        CopyTable* table_dev = reinterpret_cast<CopyTable*>(base + slot * kStaticTableStride);
        rc = launch_table_store(t, table_dev, (cudaStream_t)stream);
        if (rc == ESC_OK) rc = launch_copy_indirect(live->ctx, table_dev, copy_grid_blocks(t.n_tiles), (cudaStream_t)stream);
        if (rc != ESC_OK) return rc;
    }
    reset_stage_valid(live, 0);           // as esc_restore: stages are rebuilt lazily
    live->position = capsule->position;   // "rebind desc"
    return ESC_OK;
}

}  // extern "C"
