// Host side of libesc: context, named buffer sets, capsule verbs (include/esc.h).
// Every verb validates on the host first and enqueues exactly one copy-kernel launch.
#include <string.h>

#include <new>

#include "esc_internal.h"

namespace esc {

void free_plan_table(esc_ctx* ctx);   // graph.cu
thread_local int g_last_cuda_error = 0;

static inline uint64_t up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

uint64_t seg_valid(const Row& r, uint64_t P) { return r.fixed_bytes + P * r.bytes_per_token; }

int check_fit(const std::vector<Row>& rows, uint64_t P) {
    for (const Row& r : rows) {
        if (r.bytes_per_token && P > (UINT64_MAX - r.fixed_bytes) / r.bytes_per_token) return ESC_ERR_CAPACITY;
        const uint64_t sv = seg_valid(r, P);
        if (r.n_seg > 1 && sv > r.seg_stride) return ESC_ERR_CAPACITY;
        if ((uint64_t)(r.n_seg - 1) * r.seg_stride + sv > r.capacity) return ESC_ERR_CAPACITY;
    }
    return ESC_OK;
}

// Slab layout contract of include/esc.h: rows at 256-B multiples, segments at 16-B multiples.
void layout_walk(const std::vector<Row>& rows, uint64_t P, std::vector<Seg>* segs, uint64_t* slab_bytes,
                 uint64_t* payload_bytes) {
    uint64_t off = 0, payload = 0;
    if (segs) segs->clear();
    for (const Row& r : rows) {
        off = up(off, 256);
        const uint64_t sv = seg_valid(r, P);
        for (uint32_t s = 0; s < r.n_seg; ++s) {
            off = up(off, 16);
            if (segs) segs->push_back(Seg{r.base ? r.base + (uint64_t)s * r.seg_stride : nullptr, off, sv});
            off += sv;
            payload += sv;
        }
    }
    if (slab_bytes) *slab_bytes = off;
    if (payload_bytes) *payload_bytes = payload;
}

static uint64_t fnv1a(uint64_t h, const void* p, size_t n) {
    const uint8_t* b = (const uint8_t*)p;
    for (size_t i = 0; i < n; ++i) {
        h ^= b[i];
        h *= 0x100000001b3ull;
    }
    return h;
}

// The digest identifies the capsule LAYOUT (reading 16 of DESIGN.md), not the library build: its version word is the layout
// version, which changes only when the slab layout contract of include/esc.h does.
static const uint32_t kLayoutVersion = 1;

static uint64_t layout_digest(const std::vector<Row>& rows, const std::vector<std::string>& names) {
    uint64_t h = 0xcbf29ce484222325ull;
    h = fnv1a(h, &kLayoutVersion, sizeof kLayoutVersion);
    for (size_t i = 0; i < rows.size(); ++i) {
        const Row& r = rows[i];
        h = fnv1a(h, names[i].data(), names[i].size() + 1);
        h = fnv1a(h, &r.fixed_bytes, 8);
        h = fnv1a(h, &r.bytes_per_token, 8);
        h = fnv1a(h, &r.n_seg, 4);
    }
    return h;
}

const SegCache& live_segs(esc_bufset* live, uint64_t P) {
    SegCache& c = live->seg_cache;
    if (!c.valid || c.P != P) {
        layout_walk(live->rows, P, &c.segs, &c.slab_bytes, &c.payload_bytes);
        c.P = P;
        c.valid = true;
    }
    return c;
}

void build_restore_table(CopyTable* t, const std::vector<Seg>& segs, const uint8_t* slab) {
    const uint8_t* src[kCopyMaxSeg];
    uint8_t* dst[kCopyMaxSeg];
    uint64_t bytes[kCopyMaxSeg];
    const uint32_t n = (uint32_t)segs.size();   // callers check n <= kCopyMaxSeg
    for (uint32_t i = 0; i < n; ++i) {
        src[i] = slab + segs[i].slab_off;
        dst[i] = segs[i].live;
        bytes[i] = segs[i].bytes;
    }
    build_copy_table(t, src, dst, bytes, n);
}

int launch_copy_segs(const esc_ctx* ctx, const std::vector<Seg>& segs, uint8_t* slab, bool to_slab, cudaStream_t stream) {
    const uint8_t* src[kCopyMaxSeg];
    uint8_t* dst[kCopyMaxSeg];
    uint64_t bytes[kCopyMaxSeg];
    for (size_t first = 0; first < segs.size(); first += kCopyMaxSeg) {
        const uint32_t m = (uint32_t)(segs.size() - first < kCopyMaxSeg ? segs.size() - first : kCopyMaxSeg);
        for (uint32_t i = 0; i < m; ++i) {
            const Seg& sg = segs[first + i];
            src[i] = to_slab ? sg.live : slab + sg.slab_off;
            dst[i] = to_slab ? slab + sg.slab_off : sg.live;
            bytes[i] = sg.bytes;
        }
        int rc = launch_copy(ctx, src, dst, bytes, m, stream);
        if (rc != ESC_OK) return rc;
    }
    return ESC_OK;
}

// Pair a capsule with a live set: same layout digest, every valid range fits the live buffers.
static int pair_check(const esc_bufset* live, const esc_bufset* cap) {
    if (!live || !cap || live->frozen || !cap->frozen) return ESC_ERR_INVALID;
    if (live->layout_digest != cap->layout_digest || live->rows.size() != cap->rows.size()) return ESC_ERR_MISMATCH;
    return check_fit(live->rows, cap->position);
}

}  // namespace esc

using namespace esc;

extern "C" {

const char* esc_strerror(int code) {
    switch (code) {
        case ESC_OK: return "ESC_OK";
        case ESC_ERR_INVALID: return "ESC_ERR_INVALID: bad argument or handle kind";
        case ESC_ERR_UNALIGNED: return "ESC_ERR_UNALIGNED: boundary not a chunk multiple or pointer misaligned";
        case ESC_ERR_MISMATCH: return "ESC_ERR_MISMATCH: layout / prefix digest or position mismatch";
        case ESC_ERR_CAPACITY: return "ESC_ERR_CAPACITY: valid range exceeds a buffer or the slab";
        case ESC_ERR_UNSUPPORTED: return "ESC_ERR_UNSUPPORTED: shape / dtype / device not implemented";
        case ESC_ERR_CUDA: return "ESC_ERR_CUDA: a CUDA runtime call failed";
        default: return "ESC_ERR_?: unknown code";
    }
}

uint32_t esc_abi_version(void) { return ESC_ABI_VERSION; }
int esc_last_cuda_error(void) { return g_last_cuda_error; }

int esc_ctx_create(int device, esc_ctx** out_ctx) {
    if (!out_ctx || device < 0) return ESC_ERR_INVALID;
    int n = 0;
    ESC_CUDA(cudaGetDeviceCount(&n));
    if (device >= n) return cuda_fail(cudaErrorInvalidDevice);
    cudaDeviceProp p;
    ESC_CUDA(cudaGetDeviceProperties(&p, device));
    if (p.major != 10) return ESC_ERR_UNSUPPORTED;  // sm_100a SASS only, no fallback
    esc_ctx* c = new (std::nothrow) esc_ctx;
    if (!c) return ESC_ERR_INVALID;
    c->device = device;
    {   // create the device's primary context now (first use), leaving the caller's current device alone
        DeviceGuard g(c);
        cudaError_t e = g.err == cudaSuccess ? cudaFree(nullptr) : g.err;
        if (e != cudaSuccess) {
            delete c;
            return cuda_fail(e);
        }
    }
    c->sm_count = p.multiProcessorCount;
    c->l2_bytes = p.l2CacheSize;
    *out_ctx = c;
    return ESC_OK;
}

int esc_ctx_destroy(esc_ctx* ctx) {
    if (!ctx) return ESC_ERR_INVALID;
    ESC_ON_DEVICE(ctx);
    free_plan_table(ctx);   // the Graph[key] table owns its plans
    delete ctx;
    return ESC_OK;
}

int esc_ctx_sm_count(const esc_ctx* ctx, int* out_sms) {
    if (!ctx || !out_sms) return ESC_ERR_INVALID;
    *out_sms = ctx->sm_count;
    return ESC_OK;
}

int esc_bufset_create(esc_ctx* ctx, const esc_buf_desc* descs, uint32_t n_rows, esc_bufset** out_set) {
    if (!ctx || !descs || !out_set || n_rows == 0 || n_rows > ESC_MAX_ROWS) return ESC_ERR_INVALID;
    std::vector<Row> rows;
    rows.reserve(n_rows);
    auto names = std::make_shared<std::vector<std::string>>();
    names->reserve(n_rows);
    for (uint32_t i = 0; i < n_rows; ++i) {
        const esc_buf_desc& d = descs[i];
        if (!d.name || !d.dev_ptr || d.n_seg == 0 || d.reserved != 0) return ESC_ERR_INVALID;
        if (d.fixed_bytes == 0 && d.bytes_per_token == 0) return ESC_ERR_INVALID;
        if (d.n_seg > 1 && d.seg_stride == 0) return ESC_ERR_INVALID;
        Row r;
        names->push_back(d.name);
        r.base = (uint8_t*)d.dev_ptr;
        r.capacity = d.capacity_bytes;
        r.fixed_bytes = d.fixed_bytes;
        r.bytes_per_token = d.bytes_per_token;
        r.n_seg = d.n_seg;
        r.seg_stride = d.n_seg > 1 ? d.seg_stride : 0;
        rows.push_back(r);
    }
    if (check_fit(rows, 0) != ESC_OK) return ESC_ERR_CAPACITY;
    esc_bufset* s = new (std::nothrow) esc_bufset;
    if (!s) return ESC_ERR_INVALID;
    s->ctx = ctx;
    s->frozen = false;
    s->rows.swap(rows);
    s->layout_digest = layout_digest(s->rows, *names);
    s->names = names;
    s->position = ESC_POSITION_UNKNOWN;
    s->slab = nullptr;
    s->slab_host = nullptr;
    s->tier = ESC_TIER_GPU;
    s->slab_bytes = s->payload_bytes = s->chunk = s->prefix_digest = 0;
    *out_set = s;
    return ESC_OK;
}

int esc_bufset_destroy(esc_bufset* set) {
    if (!set) return ESC_ERR_INVALID;
    delete set;
    return ESC_OK;
}

int esc_bufset_layout_digest(const esc_bufset* set, uint64_t* out_digest) {
    if (!set || !out_digest) return ESC_ERR_INVALID;
    *out_digest = set->layout_digest;
    return ESC_OK;
}

int esc_bufset_set_position(esc_bufset* live, uint64_t position) {
    if (!live || live->frozen) return ESC_ERR_INVALID;
    if (position != ESC_POSITION_UNKNOWN) {
        int rc = check_fit(live->rows, position);
        if (rc != ESC_OK) return rc;
    }
    live->position = position;
    return ESC_OK;
}

int esc_bufset_get_position(const esc_bufset* set, uint64_t* out_position) {
    if (!set || !out_position) return ESC_ERR_INVALID;
    *out_position = set->position;
    return ESC_OK;
}

int esc_capsule_bytes(const esc_bufset* set, uint64_t P, uint64_t* out_slab_bytes, uint64_t* out_payload_bytes) {
    if (!set) return ESC_ERR_INVALID;
    int rc = check_fit(set->rows, P);
    if (rc != ESC_OK && !set->frozen) return rc;
    uint64_t slab = 0, payload = 0;
    layout_walk(set->rows, P, nullptr, &slab, &payload);
    if (out_slab_bytes) *out_slab_bytes = slab;
    if (out_payload_bytes) *out_payload_bytes = payload;
    return ESC_OK;
}

uint64_t esc_align_boundary(uint64_t P, uint64_t chunk) { return chunk ? (P / chunk) * chunk : P; }

int esc_snapshot(esc_bufset* live, uint64_t P, uint64_t chunk, uint64_t prefix_digest, uint32_t flags,
                 void* storage_dev, uint64_t storage_bytes, void* stream, esc_bufset** out_capsule) {
    if (!live || live->frozen || !out_capsule || !storage_dev) return ESC_ERR_INVALID;
    if (flags & ~ESC_SNAPSHOT_ALLOW_UNALIGNED) return ESC_ERR_INVALID;
    if (chunk && P % chunk != 0 && !(flags & ESC_SNAPSHOT_ALLOW_UNALIGNED)) return ESC_ERR_UNALIGNED;
    if (live->position != ESC_POSITION_UNKNOWN && live->position != P) return ESC_ERR_MISMATCH;
    if (((uintptr_t)storage_dev & 255u) != 0) return ESC_ERR_UNALIGNED;
    int rc = check_fit(live->rows, P);
    if (rc != ESC_OK) return rc;
    ESC_ON_DEVICE(live->ctx);
    const SegCache& sc = live_segs(live, P);
    if (sc.slab_bytes > storage_bytes) return ESC_ERR_CAPACITY;

    esc_bufset* cap = new (std::nothrow) esc_bufset;
    if (!cap) return ESC_ERR_INVALID;
    cap->ctx = live->ctx;
    cap->frozen = true;
    cap->rows = live->rows;       // plain data; the names are shared, not copied
    cap->names = live->names;
    for (Row& r : cap->rows) {   // a capsule carries the layout (and the stages' valid ends), not the live pointers
        r.base = nullptr;
        r.stage = nullptr;
    }
    cap->layout_digest = live->layout_digest;
    cap->position = P;
    cap->slab = (uint8_t*)storage_dev;
    cap->slab_host = nullptr;
    cap->tier = ESC_TIER_GPU;
    cap->slab_bytes = sc.slab_bytes;
    cap->payload_bytes = sc.payload_bytes;
    cap->chunk = chunk;
    cap->prefix_digest = prefix_digest;

    rc = launch_copy_segs(live->ctx, sc.segs, cap->slab, true, (cudaStream_t)stream);
    if (rc != ESC_OK) {
        delete cap;
        return rc;
    }
    *out_capsule = cap;
    return ESC_OK;
}

static int restore_impl(esc_bufset* live, const esc_bufset* cap, cudaStream_t stream, bool eager_dequant = false) {
    ESC_ON_DEVICE(live->ctx);
    const std::vector<Seg>& segs = live_segs(live, cap->position).segs;
    int rc;
    if (!eager_dequant) {
        rc = launch_copy_segs(live->ctx, segs, cap->slab, false, stream);
        if (rc == ESC_OK) reset_stage_valid(live, 0);   // "rebuilt lazily on the next read, not eagerly in restore"
    } else {
        std::vector<const uint8_t*> src(segs.size());
        std::vector<uint8_t*> dst(segs.size());
        std::vector<uint64_t> bytes(segs.size());
        for (size_t i = 0; i < segs.size(); ++i) {
            src[i] = cap->slab + segs[i].slab_off;
            dst[i] = segs[i].live;
            bytes[i] = segs[i].bytes;
        }
        // same walk order as layout_walk: rows in table order, segments inside a row
        std::vector<uint8_t*> d16(segs.size(), nullptr);
        std::vector<float> scale(segs.size(), 1.f);
        size_t i = 0;
        for (const Row& r : live->rows)
            for (uint32_t sg = 0; sg < r.n_seg; ++sg, ++i)
                if (r.stage) {
                    d16[i] = r.stage + 2 * ((uint64_t)sg * r.seg_stride);
                    scale[i] = r.stage_scale;
                }
        rc = launch_stage(live->ctx, src.data(), dst.data(), d16.data(), bytes.data(), scale.data(), (uint32_t)segs.size(), stream);
        if (rc == ESC_OK) reset_stage_valid(live, cap->position);
    }
    if (rc == ESC_OK) live->position = cap->position;  // "rebind desc"
    return rc;
}

int esc_restore(esc_bufset* live, const esc_bufset* capsule, const uint64_t* expect_prefix_digest, void* stream) {
    int rc = pair_check(live, capsule);
    if (rc != ESC_OK) return rc;
    if (expect_prefix_digest && *expect_prefix_digest != capsule->prefix_digest) return ESC_ERR_MISMATCH;
    return restore_impl(live, capsule, (cudaStream_t)stream);
}

int esc_restore_ex(esc_bufset* live, const esc_bufset* capsule, const uint64_t* expect_prefix_digest, uint32_t flags,
                   void* stream) {
    if (flags & ~ESC_RESTORE_DEQUANT_EAGER) return ESC_ERR_INVALID;
    int rc = pair_check(live, capsule);
    if (rc != ESC_OK) return rc;
    if (expect_prefix_digest && *expect_prefix_digest != capsule->prefix_digest) return ESC_ERR_MISMATCH;
    return restore_impl(live, capsule, (cudaStream_t)stream, (flags & ESC_RESTORE_DEQUANT_EAGER) != 0);
}

int esc_rollback(esc_bufset* live, const esc_bufset* capsule_earlier, void* stream) {
    int rc = pair_check(live, capsule_earlier);
    if (rc != ESC_OK) return rc;
    if (live->position != ESC_POSITION_UNKNOWN && live->position < capsule_earlier->position) return ESC_ERR_MISMATCH;
    return restore_impl(live, capsule_earlier, (cudaStream_t)stream);
}

int esc_fork(const esc_bufset* capsule, esc_bufset* const* lives, uint32_t n, void* stream) {
    if (!capsule || !lives || n == 0 || n > ESC_MAX_FORK) return ESC_ERR_INVALID;
    for (uint32_t d = 0; d < n; ++d) {
        int rc = pair_check(lives[d], capsule);
        if (rc != ESC_OK) return rc;
        for (uint32_t e = 0; e < d; ++e)
            if (lives[e] == lives[d]) return ESC_ERR_INVALID;
    }
    ESC_ON_DEVICE(capsule->ctx);
    std::vector<const std::vector<Seg>*> segp(n);
    for (uint32_t d = 0; d < n; ++d) segp[d] = &live_segs(lives[d], capsule->position).segs;
    const size_t ns = segp[0]->size();
    std::vector<const uint8_t*> src(ns);
    std::vector<uint64_t> bytes(ns);
    std::vector<std::vector<uint8_t*>> dst(n, std::vector<uint8_t*>(ns));
    std::vector<uint8_t* const*> dstp(n);
    for (size_t i = 0; i < ns; ++i) {
        src[i] = capsule->slab + (*segp[0])[i].slab_off;
        bytes[i] = (*segp[0])[i].bytes;
        for (uint32_t d = 0; d < n; ++d) dst[d][i] = (*segp[d])[i].live;
    }
    for (uint32_t d = 0; d < n; ++d) dstp[d] = dst[d].data();
    int rc = launch_fork(capsule->ctx, src.data(), dstp.data(), n, bytes.data(), (uint32_t)ns, (cudaStream_t)stream);
    if (rc == ESC_OK)
        for (uint32_t d = 0; d < n; ++d) {
            lives[d]->position = capsule->position;
            reset_stage_valid(lives[d], 0);
        }
    return rc;
}

int esc_capsule_info_get(const esc_bufset* capsule, esc_capsule_info* out_info) {
    if (!capsule || !capsule->frozen || !out_info) return ESC_ERR_INVALID;
    memset(out_info, 0, sizeof *out_info);
    out_info->boundary = capsule->position;
    out_info->chunk = capsule->chunk;
    out_info->slab_bytes = capsule->slab_bytes;
    out_info->payload_bytes = capsule->payload_bytes;
    out_info->layout_digest = capsule->layout_digest;
    out_info->prefix_digest = capsule->prefix_digest;
    out_info->n_rows = (uint32_t)capsule->rows.size();
    uint32_t ns = 0;
    for (const Row& r : capsule->rows) ns += r.n_seg;
    out_info->n_segments = ns;
    out_info->aligned = (capsule->chunk == 0 || capsule->position % capsule->chunk == 0) ? 1u : 0u;
    out_info->tier = capsule->tier;
    return ESC_OK;
}

// ---- tiers: a capsule slab is one contiguous range, a tier move is one async copy ----
static esc_bufset* clone_capsule(const esc_bufset* c) {
    esc_bufset* n = new (std::nothrow) esc_bufset(*c);
    return n;
}

int esc_capsule_demote(const esc_bufset* capsule, void* storage_host, uint64_t storage_bytes, void* stream,
                       esc_bufset** out_host_capsule) {
    if (!capsule || !capsule->frozen || capsule->tier != ESC_TIER_GPU || !storage_host || !out_host_capsule)
        return ESC_ERR_INVALID;
    if (storage_bytes < capsule->slab_bytes) return ESC_ERR_CAPACITY;
    if (((uintptr_t)storage_host & 255u) != 0) return ESC_ERR_UNALIGNED;
    ESC_ON_DEVICE(capsule->ctx);
    // the storage must be pinned and mapped: the restore kernels read it in place
    cudaPointerAttributes at;
    ESC_CUDA(cudaPointerGetAttributes(&at, storage_host));
    if (at.type != cudaMemoryTypeHost || !at.devicePointer) return ESC_ERR_INVALID;
    esc_bufset* h = clone_capsule(capsule);
    if (!h) return ESC_ERR_INVALID;
    h->tier = ESC_TIER_HOST;
    h->slab_host = (uint8_t*)storage_host;
    h->slab = (uint8_t*)at.devicePointer;
    cudaError_t e = capsule->slab_bytes
                        ? cudaMemcpyAsync(storage_host, capsule->slab, capsule->slab_bytes, cudaMemcpyDeviceToHost, (cudaStream_t)stream)
                        : cudaSuccess;
    if (e != cudaSuccess) {
        delete h;
        return cuda_fail(e);
    }
    *out_host_capsule = h;
    return ESC_OK;
}

int esc_capsule_promote(const esc_bufset* host_capsule, void* storage_dev, uint64_t storage_bytes, void* stream,
                        esc_bufset** out_capsule) {
    if (!host_capsule || !host_capsule->frozen || host_capsule->tier != ESC_TIER_HOST || !storage_dev || !out_capsule)
        return ESC_ERR_INVALID;
    if (storage_bytes < host_capsule->slab_bytes) return ESC_ERR_CAPACITY;
    if (((uintptr_t)storage_dev & 255u) != 0) return ESC_ERR_UNALIGNED;
    ESC_ON_DEVICE(host_capsule->ctx);
    cudaPointerAttributes at;
    ESC_CUDA(cudaPointerGetAttributes(&at, storage_dev));
    if (at.type != cudaMemoryTypeDevice) return ESC_ERR_INVALID;
    esc_bufset* g = clone_capsule(host_capsule);
    if (!g) return ESC_ERR_INVALID;
    g->tier = ESC_TIER_GPU;
    g->slab_host = nullptr;
    g->slab = (uint8_t*)storage_dev;
    cudaError_t e = host_capsule->slab_bytes ? cudaMemcpyAsync(storage_dev, host_capsule->slab_host, host_capsule->slab_bytes,
                                                               cudaMemcpyHostToDevice, (cudaStream_t)stream)
                                             : cudaSuccess;
    if (e != cudaSuccess) {
        delete g;
        return cuda_fail(e);
    }
    *out_capsule = g;
    return ESC_OK;
}

int esc_capsule_valid_end(const esc_bufset* capsule, uint32_t row, uint64_t* out_bytes_per_segment) {
    if (!capsule || !capsule->frozen || !out_bytes_per_segment || row >= capsule->rows.size()) return ESC_ERR_INVALID;
    *out_bytes_per_segment = seg_valid(capsule->rows[row], capsule->position);
    return ESC_OK;
}

}  // extern "C"
