// Host side of esc_linattn_scan (include/esc.h): shape key, argument checks, dispatch to the sm_100a
// tensor-core kernel in scan_kernel.cu.  There is one scan kernel and no fallback.
#include "esc_internal.h"

namespace esc {

// ---- host ---------------------------------------------------------------------------------------
// key layout (opaque to callers): [63:56]=0xE5 tag, B:16, H:12, dk:8(/8), dv:8(/8), in:2, out:2, chunk:8(/8)
static const uint64_t kKeyTag = 0xE5ull;

bool decode_key(esc_shape_key key, ScanShape* s) {
    if ((key >> 56) != kKeyTag) return false;
    s->B = (uint32_t)((key >> 40) & 0xFFFF);
    s->H = (uint32_t)((key >> 28) & 0xFFF);
    s->dk = (uint32_t)((key >> 20) & 0xFF) * 8;
    s->dv = (uint32_t)((key >> 12) & 0xFF) * 8;
    s->in_dtype = (uint32_t)((key >> 10) & 3);
    s->out_dtype = (uint32_t)((key >> 8) & 3);
    s->chunk = (uint32_t)(key & 0xFF) * 8;
    return true;
}

int launch_scan_tc(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g, const float* state_in,
                   float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream);

int launch_scan(esc_ctx* ctx, const ScanShape& s, const void* q, const void* k, const void* v, const float* g,
                const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride, cudaStream_t stream) {
    return launch_scan_tc(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, stream);
}

}  // namespace esc

using namespace esc;

extern "C" {

esc_shape_key esc_shape_key_make(uint32_t B, uint32_t H, uint32_t d_k, uint32_t d_v, uint32_t in_dtype,
                                 uint32_t out_dtype, uint32_t chunk) {
    if (B == 0 || H == 0 || B > 0xFFFF || H > 0xFFF || (uint64_t)B * H > 65535) return 0;
    if (!(d_k == 64 || d_k == 128) || !(d_v == 64 || d_v == 128)) return 0;
    if (!(chunk == 64 || chunk == 128)) return 0;
    if (in_dtype != ESC_DTYPE_BF16) return 0;
    if (!(out_dtype == ESC_DTYPE_F32 || out_dtype == ESC_DTYPE_BF16)) return 0;
    return (kKeyTag << 56) | ((uint64_t)B << 40) | ((uint64_t)H << 28) | ((uint64_t)(d_k / 8) << 20) |
           ((uint64_t)(d_v / 8) << 12) | ((uint64_t)in_dtype << 10) | ((uint64_t)out_dtype << 8) | (uint64_t)(chunk / 8);
}

int esc_scan_tile_columns(const esc_ctx* ctx, esc_shape_key key, uint32_t* out_columns) {
    ScanShape s;
    if (!ctx || !out_columns || !decode_key(key, &s)) return ESC_ERR_INVALID;
    *out_columns = scan_tile_columns(ctx, s);
    return ESC_OK;
}

int esc_linattn_scan(esc_ctx* ctx, esc_shape_key key, const void* q, const void* k, const void* v, const float* g,
                     const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride, uint32_t chunk,
                     void* stream) {
    ScanShape s;
    if (!ctx || !decode_key(key, &s)) return ESC_ERR_INVALID;
    if (!state_out) return ESC_ERR_INVALID;
    if (T > 0 && (!q || !k || !v || !g || !o)) return ESC_ERR_INVALID;
    if (chunk != s.chunk) return ESC_ERR_MISMATCH;
    if (t_stride < T) return ESC_ERR_INVALID;
    const uintptr_t all = (uintptr_t)q | (uintptr_t)k | (uintptr_t)v | (uintptr_t)state_in | (uintptr_t)state_out |
                          (uintptr_t)o;
    if ((all & 15u) || ((uintptr_t)g & 3u)) return ESC_ERR_UNALIGNED;  // g is read element-wise: 4-B alignment
    ESC_ON_DEVICE(ctx);
    return launch_scan(ctx, s, q, k, v, g, state_in, state_out, o, T, t_stride, (cudaStream_t)stream);
}

}  // extern "C"
