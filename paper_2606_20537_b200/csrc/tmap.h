// Tensor-map builders shared by the tensor-core scan kernels (defined in scan_kernel.cu).
#pragma once
#include <cuda.h>
#include <stdint.h>

namespace esc {

// 4-D map over a [B, t_stride, H, D] bf16 tensor whose first `T` tokens per batch row are valid:
// dims (D, H, T, B), box (box_d, 1, box_t, 1).  Rows beyond T read as zero (the short last chunk).
int make_tmap(CUtensorMap* m, const void* base, uint32_t D, uint32_t H, uint64_t T, uint64_t t_stride, uint32_t B, uint32_t box_d,
              uint32_t box_t, CUtensorMapSwizzle sw);
// whole [box_t x D] tiles as 64-column halves, 128-byte swizzle: dims (d % 64, t, d / 64, h, b), box (64, box_t, D / 64, 1, 1)
int make_tmap_halves(CUtensorMap* m, const void* base, uint32_t D, uint32_t H, uint64_t T, uint64_t t_stride, uint32_t B, uint32_t box_t);

}  // namespace esc
