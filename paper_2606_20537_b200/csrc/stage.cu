// FP8 (E4M3) KV rows and their BF16 dequantisation stage (include/esc.h; reading 23).
//
// One kernel serves the lazy rebuild (esc_dequant_stage_fill: live FP8 row -> stage) and the eager, fused restore
// (esc_restore_ex: capsule slab -> live row AND stage, plain rows copied alongside, ONE launch).  Like the capsule
// copy kernel it is driven by a table of (row, segment) entries cut into 8 KiB tiles of source bytes, one CTA per
// tile; a thread loads 4 x 8 codes (all four loads before the first store), stores them (when the entry has an FP8
// destination) and stores 4 x 16 B of BF16, so every load / store instruction of a warp covers one contiguous
// 256 B / 512 B range (r01u: with 16-code loads each thread's 32 B of BF16 went out as two 16-byte stores at a
// 32-byte stride, half-used sectors per instruction: stage fill 17.6 -> 13.4 us, eager fused restore 27.6 -> 22.7 us).
// Roofline: HBM.  Algorithmic bytes per FP8 element: 1 read + 2 written for a fill, 1 + 1 + 2 for a fused restore.
// Arithmetic per element (the precision both sides take the rounding decisions in): cvt e4m3 -> f16 (exact) -> f32
// (exact), one fp32 multiply by the row scale, cvt.rn to bf16; NaN codes are replaced by 0x7FC0 | sign.
// The NaN replacement per code (compare, select, sign insertion) made the kernel ALU-bound (r02 ncu: ALU pipe 81 % busy, 4.9
// warps per issue stalled on the math pipe, 14.4 us per fill of 24 Mi codes); a quantised KV cache holds no NaN code, so a
// vector of eight codes is tested once (SWAR) and takes the short conversion when it has none: 9.3-10.4 us with the source
// rows L2-resident behind a restore.  (With uniformly random BYTES 6 % of the vectors have a NaN code and most warps run both
// paths: 15.5-16.4 us; bench.py fills the KV rows with the codes of normal values, the tests with every code.)
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_fp8.h>
#include <string.h>

#include "esc_internal.h"
#include "sm100_ptx.cuh"

namespace esc {

constexpr uint32_t kStageMaxSeg = 96;
constexpr uint32_t kStageUnroll = 4;                              // 8-byte code vectors in flight per thread
constexpr uint32_t kStageTile = kCopyThreads * kStageUnroll * 8u;   // 8 KiB of source bytes

struct StageTable {
    uint32_t n_seg;
    uint32_t n_tiles;
    uint32_t tile_begin[kStageMaxSeg + 1];
    uint32_t pad_;
    const uint8_t* src[kStageMaxSeg];
    uint8_t* dst8[kStageMaxSeg];     // FP8 destination (fused restore) or NULL (fill)
    uint8_t* dst16[kStageMaxSeg];    // BF16 stage or NULL (a plain row copied alongside)
    uint64_t bytes[kStageMaxSeg];
    float scale[kStageMaxSeg];
};

// two E4M3 codes (low byte = element 0) -> two bf16 (low half = element 0)
__device__ __forceinline__ uint32_t expand2(uint32_t codes, float scale) {
    const __half2_raw h = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)(codes & 0xFFFFu), __NV_E4M3);
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&h));
    const __nv_bfloat162 b = __floats2bfloat162_rn(f.x * scale, f.y * scale);
    uint32_t r = *reinterpret_cast<const uint32_t*>(&b);
    if ((codes & 0x7Fu) == 0x7Fu) r = (r & 0xFFFF0000u) | 0x7FC0u | ((codes & 0x80u) << 8);
    if ((codes & 0x7F00u) == 0x7F00u) r = (r & 0x0000FFFFu) | ((0x7FC0u | (codes & 0x8000u)) << 16);
    return r;
}

// the same for a pair without a NaN code: no fix-up, the two products as one packed multiply (same roundings)
__device__ __forceinline__ uint32_t expand2_finite(uint32_t codes, float scale) {
    const __half2_raw h = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)(codes & 0xFFFFu), __NV_E4M3);
    const float2 f = fmul2(__half22float2(*reinterpret_cast<const __half2*>(&h)), make_float2(scale, scale));
    const __nv_bfloat162 b = __floats2bfloat162_rn(f.x, f.y);
    return *reinterpret_cast<const uint32_t*>(&b);
}

// eight codes per thread: a warp loads 256 contiguous bytes and stores 512 contiguous bytes of BF16 per instruction
__device__ __forceinline__ uint2 ld_codes8(const uint2* p) {
    uint2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void put_codes8(uint8_t* d8, uint8_t* d16, uint32_t i, const uint2& v, float scale) {
    if (d8) reinterpret_cast<uint2*>(d8)[i] = v;
    if (d16) {
        // a byte is a NaN code (0x7F / 0xFF) iff (byte & 0x7F) + 1 carries into bit 7: one test for all eight codes.  The per-code
        // NaN fix-up made the kernel ALU-bound (r02 ncu: ALU pipe 81 % busy, 4.9 warps per issue stalled on the math pipe); NaN
        // codes are rare, the vectors without one take the short path.
        const uint32_t n0 = (v.x & 0x7F7F7F7Fu) + 0x01010101u, n1 = (v.y & 0x7F7F7F7Fu) + 0x01010101u;
        uint4 o;
        if (((n0 | n1) & 0x80808080u) == 0u) {
            o.x = expand2_finite(v.x, scale); o.y = expand2_finite(v.x >> 16, scale);
            o.z = expand2_finite(v.y, scale); o.w = expand2_finite(v.y >> 16, scale);
        } else {
            o.x = expand2(v.x, scale); o.y = expand2(v.x >> 16, scale);
            o.z = expand2(v.y, scale); o.w = expand2(v.y >> 16, scale);
        }
        reinterpret_cast<uint4*>(d16)[i] = o;
    }
}

__device__ __forceinline__ uint16_t expand1(uint8_t code, float scale) { return (uint16_t)(expand2(code, scale) & 0xFFFFu); }

__global__ void __launch_bounds__(kCopyThreads, 8) esc_stage_kernel(const __grid_constant__ StageTable t) {
    asm volatile("griddepcontrol.wait;" ::: "memory");   // programmatic dependent launch, as in copy_kernel.cu
    const uint32_t tid = threadIdx.x;
    for (uint32_t tile = blockIdx.x; tile < t.n_tiles; tile += gridDim.x) {
        uint32_t lo = 0, hi = t.n_seg;   // largest e with tile_begin[e] <= tile
        while (hi - lo > 1) {
            const uint32_t mid = (lo + hi) >> 1;
            if (t.tile_begin[mid] <= tile) lo = mid;
            else hi = mid;
        }
        const uint32_t e = lo;
        const uint64_t off = (uint64_t)(tile - t.tile_begin[e]) * kStageTile;
        const uint64_t left = t.bytes[e] - off;
        const uint32_t n = (uint32_t)(left < kStageTile ? left : kStageTile);
        const uint8_t* src = t.src[e] + off;
        uint8_t* d8 = t.dst8[e] ? t.dst8[e] + off : nullptr;
        uint8_t* d16 = t.dst16[e] ? t.dst16[e] + 2 * off : nullptr;
        const float scale = t.scale[e];
        const bool aligned = ((((uintptr_t)src) | ((uintptr_t)d8) | ((uintptr_t)d16)) & 15u) == 0;
        uint32_t done = 0;
        if (aligned && n == kStageTile) {   // full tile: all loads of a thread first, then its stores
            uint2 v[kStageUnroll];
#pragma unroll
            for (int u = 0; u < (int)kStageUnroll; ++u) v[u] = ld_codes8(reinterpret_cast<const uint2*>(src) + tid + u * kCopyThreads);
#pragma unroll
            for (int u = 0; u < (int)kStageUnroll; ++u) put_codes8(d8, d16, tid + u * kCopyThreads, v[u], scale);
            done = n;
        } else if (aligned) {
            const uint32_t n8 = n >> 3;
            for (uint32_t i = tid; i < n8; i += kCopyThreads) put_codes8(d8, d16, i, ld_codes8(reinterpret_cast<const uint2*>(src) + i), scale);
            done = n8 << 3;
        }
        for (uint32_t i = done + tid; i < n; i += kCopyThreads) {   // tails and unaligned pointers: element by element
            const uint8_t c = src[i];
            if (d8) d8[i] = c;
            if (d16) reinterpret_cast<uint16_t*>(d16)[i] = expand1(c, scale);
        }
    }
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

int launch_stage(const esc_ctx* ctx, const uint8_t* const* src, uint8_t* const* dst8, uint8_t* const* dst16,
                 const uint64_t* bytes, const float* scale, uint32_t n, cudaStream_t stream) {
    (void)ctx;
    for (uint32_t first = 0; first < n; first += kStageMaxSeg) {
        const uint32_t m = n - first < kStageMaxSeg ? n - first : kStageMaxSeg;
        StageTable t;
        memset(&t, 0, sizeof t);
        t.n_seg = m;
        uint64_t tiles = 0;
        for (uint32_t i = 0; i < m; ++i) {
            t.tile_begin[i] = (uint32_t)tiles;
            tiles += (bytes[first + i] + kStageTile - 1) / kStageTile;
            t.src[i] = src[first + i];
            t.dst8[i] = dst8[first + i];
            t.dst16[i] = dst16[first + i];
            t.bytes[i] = bytes[first + i];
            t.scale[i] = scale[first + i];
        }
        t.tile_begin[m] = (uint32_t)tiles;
        t.n_tiles = (uint32_t)tiles;
        if (tiles == 0) continue;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(copy_grid_blocks(tiles));
        cfg.blockDim = dim3(kCopyThreads);
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        memset(attr, 0, sizeof attr);
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        ESC_CUDA(cudaLaunchKernelEx(&cfg, esc_stage_kernel, t));
    }
    return ESC_OK;
}

void reset_stage_valid(esc_bufset* live, uint64_t tokens) {
    for (Row& r : live->rows)
        if (r.stage) r.stage_valid_tokens = tokens;
}

}  // namespace esc

using namespace esc;

extern "C" {

int esc_bufset_attach_dequant_stage(esc_bufset* live, uint32_t row, void* stage_dev, uint64_t stage_capacity_bytes,
                                    uint32_t format, float scale) {
    if (!live || live->frozen || row >= live->rows.size() || !stage_dev) return ESC_ERR_INVALID;
    if (format != ESC_FORMAT_FP8_E4M3) return ESC_ERR_UNSUPPORTED;
    Row& r = live->rows[row];
    if (r.fixed_bytes != 0 || r.bytes_per_token == 0) return ESC_ERR_INVALID;   // a pure per-token (KV) row
    if (!(scale == scale) || scale == 0.f) return ESC_ERR_INVALID;
    if (stage_capacity_bytes / 2 < r.capacity) return ESC_ERR_CAPACITY;
    if ((uintptr_t)stage_dev & 1u) return ESC_ERR_UNALIGNED;
    r.stage = (uint8_t*)stage_dev;
    r.stage_format = format;
    r.stage_scale = scale;
    r.stage_valid_tokens = 0;
    return ESC_OK;
}

int esc_dequant_stage_valid_end(const esc_bufset* set, uint32_t row, uint64_t* out_tokens) {
    if (!set || !out_tokens || row >= set->rows.size()) return ESC_ERR_INVALID;
    if (!set->rows[row].stage_format) return ESC_ERR_INVALID;
    *out_tokens = set->rows[row].stage_valid_tokens;
    return ESC_OK;
}

int esc_dequant_stage_fill(esc_bufset* live, uint32_t row, uint64_t upto_tokens, void* stream) {
    if (!live || live->frozen || (row != ESC_ALL_ROWS && row >= live->rows.size())) return ESC_ERR_INVALID;
    if (live->position != ESC_POSITION_UNKNOWN && upto_tokens > live->position) return ESC_ERR_MISMATCH;
    std::vector<Row*> todo;
    for (size_t i = 0; i < live->rows.size(); ++i)
        if ((row == ESC_ALL_ROWS || row == i) && live->rows[i].stage) todo.push_back(&live->rows[i]);
    if (todo.empty()) return ESC_ERR_INVALID;   // no stage attached
    for (Row* r : todo) {
        std::vector<Row> one(1, *r);
        int rc = check_fit(one, upto_tokens);
        if (rc != ESC_OK) return rc;
    }
    std::vector<const uint8_t*> src;
    std::vector<uint8_t*> d8, d16;
    std::vector<uint64_t> bytes;
    std::vector<float> scale;
    for (Row* r : todo) {
        const uint64_t from = r->stage_valid_tokens;
        if (upto_tokens <= from) continue;   // already in sync
        for (uint32_t s = 0; s < r->n_seg; ++s) {
            src.push_back(r->base + (uint64_t)s * r->seg_stride + from * r->bytes_per_token);
            d8.push_back(nullptr);
            d16.push_back(r->stage + 2 * ((uint64_t)s * r->seg_stride + from * r->bytes_per_token));
            bytes.push_back((upto_tokens - from) * r->bytes_per_token);
            scale.push_back(r->stage_scale);
        }
    }
    if (src.empty()) return ESC_OK;
    ESC_ON_DEVICE(live->ctx);
    int rc = launch_stage(live->ctx, src.data(), d8.data(), d16.data(), bytes.data(), scale.data(), (uint32_t)src.size(),
                          (cudaStream_t)stream);
    if (rc == ESC_OK)
        for (Row* r : todo)
            if (r->stage_valid_tokens < upto_tokens) r->stage_valid_tokens = upto_tokens;
    return rc;
}

}  // extern "C"
