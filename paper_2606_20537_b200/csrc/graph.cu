// Captured replay plan: [restore node] -> [scan node per layer] as ONE CUDA graph
// (include/esc.h: esc_graph_*).  PAPER.md:128-129: restore "replay[s] the already-captured
// Graph[key] — never a recapture"; the host overwrites a bound sub-buffer between
// replays.  Here the bound sub-buffer is the restore node's copy table: it lives in a small
// caller-owned device scratch buffer (esc_graph_scratch_bytes), and binding another capsule is one
// one-CTA kernel that stores the new table there (the table travels as a kernel parameter: no copy
// engine, no host-side wait); the graph's kernel nodes (pointers, grids) never change.
#include <string.h>

#include <new>

#include "esc_internal.h"

struct esc_graph {
    esc_ctx* ctx;
    esc_bufset* live;             // NULL: cold plan (no restore node)
    cudaGraph_t graph;
    cudaGraphExec_t exec;
    esc::CopyTable* table_dev;    // device-resident "current capsule" table in the CALLER's scratch (rewritten by launch_table_store)
    bool bound;
    bool owned_by_table;          // held by the context's Graph[key] table: only the table may destroy it
    uint64_t bound_boundary;
    uint64_t max_boundary;        // the restore node's grid covers capsules up to this boundary
};

using namespace esc;

static void graph_free(esc_graph* g);
namespace esc {
void free_plan_table(esc_ctx* ctx) {
    for (auto& e : ctx->plans) graph_free(e.second);
    ctx->plans.clear();
}
}  // namespace esc

static void graph_free(esc_graph* g) {
    if (!g) return;
    if (g->exec) cudaGraphExecDestroy(g->exec);
    if (g->graph) cudaGraphDestroy(g->graph);
    delete g;                     // the table lives in caller-owned scratch: nothing to free on the device
}

extern "C" {

uint64_t esc_graph_scratch_bytes(void) { return sizeof(CopyTable); }

int esc_graph_capture(esc_ctx* ctx, esc_bufset* live, uint64_t max_boundary, const esc_scan_args* layers,
                      uint32_t n_layers, void* scratch_dev, uint64_t scratch_bytes, void* stream, esc_graph** out_graph) {
    if (!ctx || !out_graph || (n_layers && !layers) || (!live && n_layers == 0)) return ESC_ERR_INVALID;
    if (!stream) return ESC_ERR_INVALID;  // the legacy default stream cannot be captured
    if (live && (live->frozen || live->ctx != ctx)) return ESC_ERR_INVALID;
    if (live) {   // the restore node's table lives in the caller's scratch
        if (!scratch_dev) return ESC_ERR_INVALID;
        if ((uintptr_t)scratch_dev & 15u) return ESC_ERR_UNALIGNED;
        if (scratch_bytes < sizeof(CopyTable)) return ESC_ERR_CAPACITY;
    }
    ESC_ON_DEVICE(ctx);
    uint32_t grid = 0;
    if (live) {
        int rc = check_fit(live->rows, max_boundary);
        if (rc != ESC_OK) return rc;
        std::vector<Seg> segs;
        layout_walk(live->rows, max_boundary, &segs, nullptr, nullptr);
        if (segs.size() > kCopyMaxSeg) return ESC_ERR_UNSUPPORTED;
        uint64_t tiles = 0;
        for (const Seg& s : segs) tiles += (s.bytes + kCopyTileBytes - 1) / kCopyTileBytes;
        grid = copy_grid_blocks(tiles);   // one CTA per tile at max_boundary; CTAs beyond the bound capsule's tiles exit
    }
    // validate the scan layers and set kernel attributes BEFORE the capture begins
    std::vector<ScanShape> shapes(n_layers);
    for (uint32_t i = 0; i < n_layers; ++i) {
        const esc_scan_args& a = layers[i];
        if (!decode_key(a.key, &shapes[i]) || !a.state_out || a.kind > ESC_SCAN_GDN) return ESC_ERR_INVALID;
        const bool gdn = a.kind == ESC_SCAN_GDN;
        if (gdn ? (a.T > 0 && !a.beta) : a.beta != nullptr) return ESC_ERR_INVALID;
        if (gdn && shapes[i].out_dtype != ESC_DTYPE_F32) return ESC_ERR_UNSUPPORTED;
        if (a.T > 0 && (!a.q || !a.k || !a.v || !a.g || !a.o)) return ESC_ERR_INVALID;
        if (a.chunk != shapes[i].chunk) return ESC_ERR_MISMATCH;
        if (a.t_stride < a.T) return ESC_ERR_INVALID;
        const uintptr_t all = (uintptr_t)a.q | (uintptr_t)a.k | (uintptr_t)a.v | (uintptr_t)a.state_in |
                              (uintptr_t)a.state_out | (uintptr_t)a.o;
        if ((all & 15u) || (((uintptr_t)a.g | (uintptr_t)a.beta) & 3u)) return ESC_ERR_UNALIGNED;
        // prepare-only calls (state_out == NULL): kernel attributes may not be set during a capture
        int rc = gdn ? launch_gdn_mma(ctx, shapes[i], nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 0, 0, nullptr)
                     : launch_scan(ctx, shapes[i], nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 0, 0, nullptr);
        if (rc != ESC_OK) return rc;
    }

    esc_graph* g = new (std::nothrow) esc_graph();
    if (!g) return ESC_ERR_INVALID;
    g->ctx = ctx;
    g->live = live;
    g->bound = false;
    g->owned_by_table = false;
    g->max_boundary = max_boundary;
    cudaError_t e = cudaSuccess;
    cudaStream_t st = (cudaStream_t)stream;
    if (live) {
        // an empty table (n_tiles = 0: the restore node is a no-op until a capsule is bound), stored by a kernel on the
        // CALLER's stream ahead of the capture: ordered before every later launch / set_capsule on that stream, unlike a
        // memset on the legacy stream, which a non-blocking stream does not wait for
        g->table_dev = (CopyTable*)scratch_dev;
        CopyTable empty;
        memset(&empty, 0, sizeof empty);
        int rc0 = launch_table_store(empty, g->table_dev, st);
        if (rc0 != ESC_OK) {
            graph_free(g);
            return rc0;
        }
    }
    e = cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) {
        graph_free(g);
        return cuda_fail(e);
    }
    int rc = ESC_OK;
    if (live) rc = launch_copy_indirect(ctx, g->table_dev, grid, st);
    for (uint32_t i = 0; i < n_layers && rc == ESC_OK; ++i) {
        const esc_scan_args& a = layers[i];
        rc = a.kind == ESC_SCAN_GDN ? launch_gdn_mma(ctx, shapes[i], a.q, a.k, a.v, a.g, a.beta, a.state_in, a.state_out, (float*)a.o, a.T, a.t_stride, st)
                                    : launch_scan(ctx, shapes[i], a.q, a.k, a.v, a.g, a.state_in, a.state_out, a.o, a.T, a.t_stride, st);
    }
    e = cudaStreamEndCapture(st, &g->graph);
    if (rc != ESC_OK || e != cudaSuccess) {
        graph_free(g);
        return rc != ESC_OK ? rc : cuda_fail(e);
    }
    e = cudaGraphInstantiate(&g->exec, g->graph, 0);
    if (e != cudaSuccess) {
        graph_free(g);
        return cuda_fail(e);
    }
    *out_graph = g;
    return ESC_OK;
}

int esc_graph_set_capsule(esc_graph* graph, const esc_bufset* capsule, void* stream) {
    if (!graph || !graph->live || !capsule || !capsule->frozen) return ESC_ERR_INVALID;
    esc_bufset* live = graph->live;
    if (live->layout_digest != capsule->layout_digest || live->rows.size() != capsule->rows.size())
        return ESC_ERR_MISMATCH;
    if (capsule->position > graph->max_boundary) return ESC_ERR_CAPACITY;   // the plan was sized for boundaries <= max_boundary
    int rc = check_fit(live->rows, capsule->position);
    if (rc != ESC_OK) return rc;
    ESC_ON_DEVICE(graph->ctx);
    const std::vector<Seg>& segs = live_segs(live, capsule->position).segs;
    if (segs.size() > kCopyMaxSeg) return ESC_ERR_UNSUPPORTED;
    CopyTable t;
    build_restore_table(&t, segs, capsule->slab);
    rc = launch_table_store(t, graph->table_dev, (cudaStream_t)stream);
    if (rc != ESC_OK) return rc;
    graph->bound = true;
    graph->bound_boundary = capsule->position;
    return ESC_OK;
}

int esc_graph_launch(esc_graph* graph, void* stream) {
    if (!graph) return ESC_ERR_INVALID;
    if (graph->live && !graph->bound) return ESC_ERR_INVALID;
    ESC_ON_DEVICE(graph->ctx);
    ESC_CUDA(cudaGraphLaunch(graph->exec, (cudaStream_t)stream));
    if (graph->live) {
        graph->live->position = graph->bound_boundary;
        reset_stage_valid(graph->live, 0);   // the restore node copies FP8 rows only: stages are rebuilt lazily
    }
    return ESC_OK;
}

int esc_graph_destroy(esc_graph* graph) {
    if (!graph) return ESC_ERR_INVALID;
    if (graph->owned_by_table) return ESC_ERR_INVALID;   // the Graph[key] table owns it (evicts / destroys it itself)
    ESC_ON_DEVICE(graph->ctx);
    graph_free(graph);
    return ESC_OK;
}

// ---- Graph[key] table: bounded, LRU ------------------------------------------------
uint64_t esc_suffix_bucket(uint64_t T, uint64_t chunk) {
    if (T == 0 || chunk == 0) return T;
    uint64_t b = chunk;
    while (b < T && b <= (UINT64_MAX >> 1)) b <<= 1;
    return b;
}

uint64_t esc_plan_key_make(esc_shape_key key, uint64_t suffix_bucket, uint64_t max_boundary, uint32_t n_layers) {
    uint64_t h = 0xcbf29ce484222325ull;
    const uint64_t v[4] = {key, suffix_bucket, max_boundary, n_layers};
    const uint8_t* b = (const uint8_t*)v;
    for (size_t i = 0; i < sizeof v; ++i) {
        h ^= b[i];
        h *= 0x100000001b3ull;
    }
    return h;
}

static void plan_evict_to(esc_ctx* ctx, size_t n) {
    DeviceGuard g(ctx);
    while (ctx->plans.size() > n) {
        graph_free(ctx->plans.back().second);
        ctx->plans.pop_back();
        ++ctx->plan_evictions;
    }
}

int esc_plan_table_set_capacity(esc_ctx* ctx, uint32_t capacity) {
    if (!ctx || capacity == 0) return ESC_ERR_INVALID;
    ctx->plan_capacity = capacity;
    plan_evict_to(ctx, capacity);
    return ESC_OK;
}

int esc_plan_table_put(esc_ctx* ctx, uint64_t plan_key, esc_graph* graph) {
    if (!ctx || !graph || graph->ctx != ctx) return ESC_ERR_INVALID;
    // a plan is owned once: the whole table is searched for the handle before anything changes
    for (size_t i = 0; i < ctx->plans.size(); ++i)
        if (ctx->plans[i].second == graph && ctx->plans[i].first != plan_key) return ESC_ERR_INVALID;
    for (size_t i = 0; i < ctx->plans.size(); ++i)
        if (ctx->plans[i].first == plan_key) {
            if (ctx->plans[i].second != graph) {
                DeviceGuard g(ctx);
                graph_free(ctx->plans[i].second);
            }
            ctx->plans.erase(ctx->plans.begin() + i);
            break;
        }
    plan_evict_to(ctx, ctx->plan_capacity - 1);
    graph->owned_by_table = true;
    ctx->plans.insert(ctx->plans.begin(), std::make_pair(plan_key, graph));
    return ESC_OK;
}

// 1 when `plan_key` is in the table (does not touch the LRU order or the statistics): lets a binding drop its references
// to plans the table has evicted
int esc_plan_table_contains(const esc_ctx* ctx, uint64_t plan_key, uint32_t* out_present) {
    if (!ctx || !out_present) return ESC_ERR_INVALID;
    *out_present = 0;
    for (const auto& e : ctx->plans)
        if (e.first == plan_key) *out_present = 1;
    return ESC_OK;
}

int esc_plan_table_get(esc_ctx* ctx, uint64_t plan_key, esc_graph** out_graph) {
    if (!ctx || !out_graph) return ESC_ERR_INVALID;
    for (size_t i = 0; i < ctx->plans.size(); ++i)
        if (ctx->plans[i].first == plan_key) {
            std::pair<uint64_t, esc_graph*> e = ctx->plans[i];
            ctx->plans.erase(ctx->plans.begin() + i);
            ctx->plans.insert(ctx->plans.begin(), e);
            ++ctx->plan_hits;
            *out_graph = e.second;
            return ESC_OK;
        }
    ++ctx->plan_misses;
    return ESC_ERR_MISMATCH;
}

int esc_plan_table_stats(const esc_ctx* ctx, uint32_t* out_size, uint64_t* out_hits, uint64_t* out_misses,
                         uint64_t* out_evictions) {
    if (!ctx) return ESC_ERR_INVALID;
    if (out_size) *out_size = (uint32_t)ctx->plans.size();
    if (out_hits) *out_hits = ctx->plan_hits;
    if (out_misses) *out_misses = ctx->plan_misses;
    if (out_evictions) *out_evictions = ctx->plan_evictions;
    return ESC_OK;
}

}  // extern "C"
