"""Oracle of the FP8 -> BF16 dequantisation stage.

ORACLE — TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  Shares no code with the CUDA path.

PAPER.md:86: the KV region of a capsule is "the persistent full-attention KV valid over [0, P), plus the
long-context FP8 dequantization stage's valid end"; "FP8-KV roughly halves it".  PAPER.md:102: "the FP8 -> BF16
working stage is rebuilt lazily on the next read, not eagerly in restore".  The paper gives neither the FP8
format nor the scaling; reading 23 fixes them:
  * format: OCP FP8 E4M3 ("E4M3FN"): 1 sign, 4 exponent bits (bias 7), 3 mantissa bits, no infinities,
    NaN = S.1111.111, subnormals at exponent field 0;
  * stage element i = bf16_rne( fp32(decode(code_i)) * fp32(scale) ), one per-row fp32 scale; the product is
    rounded once to fp32 (IEEE multiply) and once more to bf16 (round to nearest even) — the precision the
    kernel takes the decision in; NaN codes map to the quiet NaN 0x7FC0 with the code's sign.
Written out step by step below: a 256-entry table from the format definition, then plain numpy fp32.
"""
import numpy as np


def e4m3_decode_table() -> np.ndarray:
    """float64[256]: the value of every E4M3 code, from the format definition (NaN for S.1111.111)."""
    t = np.zeros(256, dtype=np.float64)
    for code in range(256):
        sign = -1.0 if code & 0x80 else 1.0
        e = (code >> 3) & 0xF
        m = code & 0x7
        if e == 0xF and m == 0x7:
            t[code] = np.nan
        elif e == 0:
            t[code] = sign * (m / 8.0) * 2.0 ** (1 - 7)          # subnormal: 0.m x 2^(1-bias)
        else:
            t[code] = sign * (1.0 + m / 8.0) * 2.0 ** (e - 7)     # normal: 1.m x 2^(e-bias)
    return t


def f32_to_bf16_bits_rne(x: np.ndarray) -> np.ndarray:
    """uint16 bf16 bit patterns of float32 values, round to nearest even (finite inputs)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    lsb = (u >> np.uint64(16)) & np.uint64(1)
    return ((u + np.uint64(0x7FFF) + lsb) >> np.uint64(16)).astype(np.uint16)


def dequant_stage(codes: np.ndarray, scale: float) -> np.ndarray:
    """uint8 E4M3 codes (any shape) -> uint16 bf16 bit patterns of the stage elements."""
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    table = e4m3_decode_table()
    val = table[codes].astype(np.float32)                  # exact: every E4M3 value is a float32
    is_nan = np.isnan(val)
    with np.errstate(invalid="ignore"):
        prod = val * np.float32(scale)                     # one IEEE fp32 multiply
    bits = f32_to_bf16_bits_rne(np.where(is_nan, np.float32(0), prod))
    nan_bits = (np.uint16(0x7FC0) | ((codes.astype(np.uint16) & np.uint16(0x80)) << np.uint16(8))).astype(np.uint16)
    return np.where(is_nan, nan_bits, bits).astype(np.uint16)
