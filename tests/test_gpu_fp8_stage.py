"""-m gpu parity of the FP8 (E4M3) KV rows and their BF16 dequantisation stage (include/esc.h) against
oracle/fp8_stage.py: integer work, so everything is bit-exact — capsule bytes by memcmp, stage elements as uint16."""
import numpy as np
import pytest
import torch

import oracle
from oracle import fp8_stage
from paper_2606_20537_b200 import synth
from gpu_util import DEV, LiveSet, esc_mod

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def esc():
    return esc_mod()


@pytest.fixture(scope="module")
def ctx(esc):
    c = esc.Ctx(0)
    yield c
    c.close()


def _fp8_layout(t_max, head_major):
    # config-1 layer mix at reduced size with FP8 KV (1 byte per element): "FP8-KV roughly halves it"
    return synth.hybrid_layout(t_max, n_linear=3, n_full=2, H=2, dk=64, dv=64, kv_heads=2, head_dim=72, kv_elem_bytes=1,
                               head_major=head_major)


def _attach(esc, live, scales, offset=0):
    """Attach a BF16 stage (filled with a 0xABAB pattern) to every KV row; returns {row: stage tensor}."""
    stages = {}
    for i, s in enumerate(live.specs):
        if s.bytes_per_token:
            base = torch.full((2 * (s.capacity_bytes + 8 + offset),), 0xAB, dtype=torch.uint8, device=DEV)
            st = base[2 * offset: 2 * offset + 2 * s.capacity_bytes]
            live.set.attach_dequant_stage(i, st, scale=scales[i % len(scales)], stage_bytes=2 * s.capacity_bytes)
            stages[i] = (st, scales[i % len(scales)])
    return stages


def _expected_stage(live, i, scale, tokens):
    """oracle: uint16 stage image of row i with tokens [0, tokens) of every segment expanded, the rest 0xABAB."""
    s = live.specs[i]
    exp = np.full(s.capacity_bytes, 0xABAB, dtype=np.uint16)
    for seg in range(s.n_seg):
        a = seg * s.seg_stride
        n = tokens * s.bytes_per_token
        exp[a:a + n] = fp8_stage.dequant_stage(live.host[i][a:a + n], scale)
    return exp


def _stage_bits(st):
    return st.cpu().numpy().view(np.uint16)


@pytest.mark.parametrize("head_major", [False, True])
def test_lazy_fill_and_eager_restore_bit_exact(esc, ctx, head_major):
    P, t_max = 300, 512        # 300 tokens x 144 B: not a tile multiple; head_dim 72: ragged 16-byte tails per segment
    specs = _fp8_layout(t_max, head_major)
    live = LiveSet(esc, ctx, specs, (7, int(head_major)))      # random bytes: every E4M3 code incl. NaN codes and -0
    scales = [1.0, 0.37, 1.0 / 448.0]
    stages = _attach(esc, live, scales)
    live.set.set_position(P)
    slab = torch.empty(live.set.capsule_bytes(P)[0], dtype=torch.uint8, device=DEV)
    # lazy fill in two steps (watermark): [0,100) then [100,P)
    rows = sorted(stages)
    for i in rows:
        assert live.set.stage_valid_end(i) == 0
        live.set.stage_fill(i, 100)
        assert live.set.stage_valid_end(i) == 100
    torch.cuda.synchronize()
    for i in rows:
        assert np.array_equal(_stage_bits(stages[i][0]), _expected_stage(live, i, stages[i][1], 100)), specs[i].name
    live.set.stage_fill(esc.ALL_ROWS, P)                        # every staged row, one launch
    cap = esc.snapshot(live.set, P, 0, slab)
    torch.cuda.synchronize()
    for i in rows:
        assert np.array_equal(_stage_bits(stages[i][0]), _expected_stage(live, i, stages[i][1], P)), specs[i].name
        assert cap.stage_valid_end(i) == P                      # the capsule records the stage's valid end
    ref_slab = oracle.capsule_snapshot(live.oracle_rows(), P)
    payload = live.set.capsule_bytes(P)[1]
    assert payload == sum(s.fixed_bytes * s.n_seg + P * s.bytes_per_token * s.n_seg for s in specs)
    # plain restore after dirtying rows AND stages: FP8 bytes back, stages untouched and marked invalid (lazy rule)
    saved = {i: live.host[i].copy() for i in range(len(specs))}
    live.fill(8, 0, pattern=0xFF)
    for i in rows:
        stages[i][0].fill_(0xCD)
    esc.restore(live.set, cap)
    oracle.capsule_restore(live.oracle_rows(), P, ref_slab)
    live.assert_equals_host()
    for i in rows:
        assert live.set.stage_valid_end(i) == 0
        assert bool((stages[i][0] == 0xCD).all())
    # eager restore: one launch restores the rows and rebuilds every stage over [0, P)
    live.fill(9, 0, pattern=0x7F)                               # 0x7F = the NaN code everywhere
    for i in rows:
        stages[i][0].fill_(0xAB)
    esc.restore_ex(live.set, cap, flags=esc.RESTORE_DEQUANT_EAGER)
    oracle.capsule_restore(live.oracle_rows(), P, ref_slab)
    live.assert_equals_host()
    for i in rows:
        assert live.set.stage_valid_end(i) == P
        assert np.array_equal(_stage_bits(stages[i][0]), _expected_stage(live, i, stages[i][1], P)), specs[i].name
    assert live.set.position == P
    cap.destroy()
    live.set.destroy()


def test_all_codes_and_unaligned_stage(esc, ctx):
    # every code value at every byte phase, stage pointer 2-byte (not 16-byte) aligned: the element path
    specs = [synth.RowSpec("L00.full.k", 4096, 0, 256, 1, 0)]
    live = LiveSet(esc, ctx, specs, (10,))
    codes = np.tile(np.arange(256, dtype=np.uint8), 16)
    live.set_row(0, codes)
    stages = _attach(esc, live, [0.0123], offset=1)
    live.set.stage_fill(0, 16)
    torch.cuda.synchronize()
    got = _stage_bits(stages[0][0])
    assert np.array_equal(got, fp8_stage.dequant_stage(codes, 0.0123))
    assert got[0x7F] == 0x7FC0 and got[0xFF] == 0xFFC0


def test_stage_errors(esc, ctx):
    specs = _fp8_layout(128, False)
    live = LiveSet(esc, ctx, specs, (11,))
    kv = [i for i, s in enumerate(specs) if s.bytes_per_token][0]
    lin = [i for i, s in enumerate(specs) if not s.bytes_per_token][0]
    st = torch.empty(2 * specs[kv].capacity_bytes, dtype=torch.uint8, device=DEV)
    for row, tensor, nbytes, fmt, scale, code in (
            (lin, st, None, esc.FORMAT_FP8_E4M3, 1.0, esc.ERR_INVALID),          # a fold state is not a per-token row
            (kv, st, specs[kv].capacity_bytes, esc.FORMAT_FP8_E4M3, 1.0, esc.ERR_CAPACITY),
            (kv, st, None, 9, 1.0, esc.ERR_UNSUPPORTED),
            (kv, st, None, esc.FORMAT_FP8_E4M3, 0.0, esc.ERR_INVALID)):
        with pytest.raises(esc.EscError) as e:
            live.set.attach_dequant_stage(row, tensor, scale=scale, fmt=fmt, stage_bytes=nbytes)
        assert e.value.code == code
    with pytest.raises(esc.EscError):
        live.set.stage_fill(kv, 10)                                               # no stage attached
    live.set.attach_dequant_stage(kv, st)
    live.set.set_position(64)
    with pytest.raises(esc.EscError) as e:
        live.set.stage_fill(kv, 65)                                               # beyond the live position
    assert e.value.code == esc.ERR_MISMATCH
    live.set.stage_fill(kv, 64)
    assert live.set.stage_valid_end(kv) == 64


def test_full_size_fp8_config1_sampled(esc, ctx):
    # config-1 geometry with FP8 KV: 18 fold states + 6 layers x (K, V) [T,4,256] E4M3: 18 MiB + 12 KiB x 2048 = 42 MiB
    P = 2048
    specs = synth.hybrid_layout(P + 64, kv_elem_bytes=1)
    g = torch.Generator(device=DEV)
    g.manual_seed(1234)
    bufs = [torch.randint(0, 256, (s.capacity_bytes,), dtype=torch.uint8, device=DEV, generator=g) for s in specs]
    live = esc.bufset_create(ctx, [(s.name, b, s.capacity_bytes, s.fixed_bytes, s.bytes_per_token, s.n_seg, s.seg_stride)
                                   for s, b in zip(specs, bufs)])
    stages = {}
    for i, s in enumerate(specs):
        if s.bytes_per_token:
            stages[i] = torch.zeros(s.capacity_bytes, dtype=torch.bfloat16, device=DEV)
            live.attach_dequant_stage(i, stages[i], scale=0.25)
    live.set_position(P)
    slab_bytes, payload = live.capsule_bytes(P)
    assert payload == 18 * (1 << 20) + 12288 * P
    slab = torch.empty(slab_bytes, dtype=torch.uint8, device=DEV)
    cap = esc.snapshot(live, P, 64, slab)
    keep = [b.clone() for b in bufs]
    for b in bufs:
        b.fill_(0xFF)
    esc.restore_ex(live, cap, flags=esc.RESTORE_DEQUANT_EAGER)
    torch.cuda.synchronize()
    for i, s in enumerate(specs):
        nv = s.fixed_bytes + P * s.bytes_per_token
        assert torch.equal(bufs[i][:nv], keep[i][:nv]), s.name
    rng = np.random.default_rng(3)
    for i in sorted(stages)[::3]:
        s = specs[i]
        for t in rng.integers(0, P, size=6):
            a = int(t) * s.bytes_per_token
            codes = keep[i][a:a + s.bytes_per_token].cpu().numpy()
            got = stages[i].view(torch.int16)[a:a + s.bytes_per_token].cpu().numpy().view(np.uint16)
            assert np.array_equal(got, fp8_stage.dequant_stage(codes, 0.25)), (s.name, int(t))
