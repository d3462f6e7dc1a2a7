"""Pins of the FP8 (E4M3) dequantisation-stage oracle against things other than itself: the format's closed
forms, torch's own float8_e4m3fn conversion (a library routine), exactness in bf16, rounding cases by hand."""
import numpy as np
import pytest
import torch

from oracle import fp8_stage


def test_table_closed_forms():
    t = fp8_stage.e4m3_decode_table()
    assert t[0x00] == 0.0 and t[0x80] == 0.0 and np.signbit(t[0x80])
    assert t[0x38] == 1.0 and t[0xB8] == -1.0                  # e = 7 (bias), m = 0
    assert t[0x7E] == 448.0                                     # largest finite: 1.75 * 2^8
    assert t[0x01] == 2.0 ** -9 and t[0x07] == 7 * 2.0 ** -9    # subnormals: m/8 * 2^-6
    assert t[0x08] == 2.0 ** -6                                 # smallest normal
    assert np.isnan(t[0x7F]) and np.isnan(t[0xFF])              # the only NaN codes; no infinities
    fin = t[:0x7F]
    assert np.all(np.diff(fin) > 0)                             # strictly increasing over the positive codes
    assert np.array_equal(t[0x80:0xFF], -t[0x00:0x7F])          # sign symmetry


def test_table_matches_torch_float8_e4m3fn():
    codes = torch.arange(256, dtype=torch.int32).to(torch.uint8)
    ref = codes.view(torch.float8_e4m3fn).to(torch.float32).numpy().astype(np.float64)
    t = fp8_stage.e4m3_decode_table()
    assert np.array_equal(np.isnan(ref), np.isnan(t))
    ok = ~np.isnan(t)
    assert np.array_equal(ref[ok], t[ok])


def test_stage_scale_one_is_exact_and_bf16_representable():
    codes = np.arange(256, dtype=np.uint8)
    bits = fp8_stage.dequant_stage(codes, 1.0)
    back = (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    t = fp8_stage.e4m3_decode_table()
    ok = ~np.isnan(t)
    assert np.array_equal(back[ok], t[ok])                      # 4 significant bits fit bf16's 8: no rounding at scale 1
    assert bits[0x7F] == 0x7FC0 and bits[0xFF] == 0xFFC0
    assert bits[0x80] == 0x8000                                 # -0 keeps its sign


def test_stage_rounding_matches_torch_bfloat16_and_hand_cases():
    rng = np.random.default_rng(5)
    codes = rng.integers(0, 256, size=4096, dtype=np.uint8)
    codes = codes[(codes & 0x7F) != 0x7F]
    for scale in (0.3, 1.0 / 448.0, 17.25, 3.0e-5):
        bits = fp8_stage.dequant_stage(codes, scale)
        v = torch.from_numpy(codes).view(torch.float8_e4m3fn).to(torch.float32) * torch.tensor(scale, dtype=torch.float32)
        ref = v.to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
        assert np.array_equal(bits, ref), scale
    # by hand: 1.0 * (1 + 2^-8) is a tie between bf16 1.0 (even) and 1.0078125 -> rounds to even = 0x3F80
    assert fp8_stage.f32_to_bf16_bits_rne(np.array([1.0 + 2.0 ** -8], np.float32))[0] == 0x3F80
    # 1 + 3 * 2^-8 is a tie between 0x3F81 (odd) and 0x3F82 (even) -> 0x3F82
    assert fp8_stage.f32_to_bf16_bits_rne(np.array([1.0 + 3 * 2.0 ** -8], np.float32))[0] == 0x3F82
    # just above a tie rounds up
    assert fp8_stage.f32_to_bf16_bits_rne(np.array([np.float32(1.0 + 2.0 ** -8 + 2.0 ** -20)], np.float32))[0] == 0x3F81
