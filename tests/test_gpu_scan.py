"""-m gpu parity tests of esc_linattn_scan through the C ABI against the fp64 sequential oracle.

Bars (BASELINE.json north_star, metric readings #7/#8 of DESIGN.md):
  o: ||o_gpu - o_ref||_inf / ||o_ref||_inf <= 2e-3 ;  S_T: relative Frobenius <= 1e-3 ;
  chunk-aligned restore + continue == cold run, bit for bit;
  bf16-o variant == RNE-bf16 of the fp32-o kernel's result, bit for bit."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_20537_b200 import synth
from gpu_util import (DEV, TOL_O, TOL_S, assert_state_close, bits_equal, err_o, err_s, esc_mod, sample_heads,
                      scan_dev_inputs, to_dev)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def esc():
    return esc_mod()


@pytest.fixture(scope="module")
def ctx(esc):
    c = esc.Ctx(0)
    yield c
    c.close()


def run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, s0=None, t0=0, n=None, out_bf16=False, t_stride=None):
    """Scan tokens [t0, t0+n) of device inputs laid out [B, t_stride, H, d]; returns (o[B,n,H,dv], S)."""
    q, k, v, g = dev_in
    t_stride = t_stride or q.shape[1]
    n = T - t0 if n is None else n
    key = esc.shape_key_make(B, H, dk, dv, esc.DTYPE_BF16, esc.DTYPE_BF16 if out_bf16 else esc.DTYPE_F32, chunk)
    assert key
    o = torch.full((B, t_stride, H, dv), float("nan"), dtype=torch.bfloat16 if out_bf16 else torch.float32, device=DEV)
    s_out = torch.full((B, H, dk, dv), float("nan"), dtype=torch.float32, device=DEV)
    esc.linattn_scan(ctx, key, q[:, t0:], k[:, t0:], v[:, t0:], g[:, t0:], s0, s_out, o[:, t0:], n, t_stride, chunk)
    torch.cuda.synchronize()
    return o[:, t0:t0 + n], s_out, o


SHAPES = [
    # B, H, dk, dv, T, chunk, gate
    (1, 2, 64, 64, 256, 64, "fast"),        # BASELINE config 0
    (2, 3, 128, 128, 300, 64, "fast"),      # several tiles + ragged tail
    (1, 2, 64, 128, 130, 128, "fast"),
    (1, 4, 128, 64, 257, 128, "fast"),
    (1, 16, 128, 128, 512, 64, "fast"),     # config-1/2 head shape
    (1, 2, 128, 128, 1024, 64, "slow"),     # slow decay: the carried state matters for many chunks
    (1, 2, 128, 128, 640, 128, "slow"),
    (1, 2, 64, 64, 256, 64, "one"),         # g == 1: plain linear attention
    (1, 1, 128, 128, 1, 64, "fast"),        # T = 1
    (1, 1, 128, 128, 63, 64, "fast"),       # T < chunk
    (2, 3, 64, 64, 128, 64, "fast"),        # two whole chunks in the cluster-free short-call variant (T <= 128), d = 64
    (1, 2, 128, 64, 100, 128, "slow"),      # ragged second chunk in the short-call variant, d_v = 64
    # the 32-column tile (B H d_v / 16 > SMs): every (d_k, cluster size) instantiation, long and short calls
    (2, 16, 128, 128, 330, 64, "slow"),     # d_k 128, clusters of 4
    (2, 16, 128, 128, 100, 64, "fast"),     #   ... cluster-free short call
    (2, 10, 64, 128, 300, 64, "slow"),      # d_k 64, clusters of 4
    (2, 20, 128, 64, 333, 128, "fast"),     # d_v 64: clusters of 2
    (2, 20, 64, 64, 200, 64, "slow"),       # d_k 64, d_v 64: clusters of 2
    (2, 20, 64, 64, 64, 64, "one"),         #   ... cluster-free short call
]


@pytest.mark.parametrize("B,H,dk,dv,T,chunk,gate", SHAPES)
@pytest.mark.parametrize("with_s0", [False, True])
def test_scan_vs_oracle(esc, ctx, B, H, dk, dv, T, chunk, gate, with_s0):
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(10, T, dk, dv), gate=gate)
    s0_np = synth.scan_state(B, H, dk, dv, seed_ids=(T,), scale=0.5) if with_s0 else None
    o_ref, s_ref = oracle.linattn_recurrence(*si.as_f32(), None if s0_np is None else s0_np.astype(np.float64))
    dev_in = scan_dev_inputs(si)
    o, s, o_full = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, None if s0_np is None else to_dev(s0_np))
    assert not torch.isnan(o).any() and not torch.isnan(s).any()
    eo = err_o(o.cpu().numpy(), o_ref)
    assert eo <= TOL_O, "o error %.3e" % eo
    assert_state_close(s, s_ref)
    # bf16-o variant: RNE of the fp32 kernel's result, state identical
    o16, s16, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, None if s0_np is None else to_dev(s0_np),
                           out_bf16=True)
    assert bits_equal(o16, o.to(torch.bfloat16)) and bits_equal(s16, s)


def test_empty_T_copies_state(esc, ctx):
    B, H, dk, dv = 1, 2, 64, 64
    si = synth.scan_inputs(B, 4, H, dk, dv, seed_ids=(11,))
    s0 = to_dev(synth.scan_state(B, H, dk, dv, seed_ids=(11,)))
    _, s, _ = run_scan(esc, ctx, scan_dev_inputs(si), B, 0, H, dk, dv, 64, s0, n=0)
    assert bits_equal(s, s0)
    _, s, _ = run_scan(esc, ctx, scan_dev_inputs(si), B, 0, H, dk, dv, 64, None, n=0)
    assert bool((s == 0).all())


def test_batch_stride_and_untouched_tail(esc, ctx):
    # only tokens [0,T) of each batch row are read / written; t_stride > T
    B, H, dk, dv, Tbuf, T = 2, 2, 64, 64, 200, 150
    si = synth.scan_inputs(B, Tbuf, H, dk, dv, seed_ids=(12,))
    o_ref, s_ref = oracle.linattn_recurrence(*si.as_f32(), T=T)
    o, s, o_full = run_scan(esc, ctx, scan_dev_inputs(si), B, T, H, dk, dv, 64, n=T)
    assert err_o(o.cpu().numpy(), o_ref) <= TOL_O
    assert_state_close(s, s_ref)
    assert torch.isnan(o_full[:, T:]).all(), "tokens beyond T were written"


@pytest.mark.parametrize("B,H,dk,dv,T,chunk,P", [
    (1, 2, 64, 64, 256, 64, 128),          # config 0: snapshot at t=128, restore, continue 128
    (2, 4, 128, 128, 448, 64, 192),
    (1, 4, 128, 128, 640, 128, 384),
    (2, 16, 128, 128, 448, 64, 192),       # 32-column tile, long continuation (clusters of 4)
    (4, 16, 128, 128, 320, 64, 256),       # 32-column tile, continuation of 64 tokens: the cluster-free launch
    (2, 20, 64, 64, 384, 128, 256),        # d = 64, clusters of 2
])
def test_aligned_restore_continue_is_bit_identical_to_cold(esc, ctx, B, H, dk, dv, T, chunk, P):
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(13, T, P))
    dev_in = scan_dev_inputs(si)
    o_cold, s_cold, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk)
    # prefill to P in a LIVE state buffer registered as a capsule row, snapshot, dirty, restore, continue
    key = esc.shape_key_make(B, H, dk, dv, esc.DTYPE_BF16, esc.DTYPE_F32, chunk)
    state = torch.zeros((B, H, dk, dv), dtype=torch.float32, device=DEV)
    nbytes = state.numel() * 4
    live = esc.bufset_create(ctx, [("L00.lin.state", state, nbytes, nbytes, 0, 1, 0)])
    q, k, v, g = dev_in
    o = torch.zeros((B, T, H, dv), dtype=torch.float32, device=DEV)
    esc.linattn_scan(ctx, key, q, k, v, g, None, state, o, P, T, chunk)
    assert esc.align_boundary(P, chunk) == P
    slab = torch.empty(live.capsule_bytes(P)[0], dtype=torch.uint8, device=DEV)
    cap = esc.snapshot(live, P, chunk, slab)
    state.fill_(float("nan"))                       # dirty the live fold state
    o[:, P:].fill_(float("nan"))
    esc.restore(live, cap)
    esc.linattn_scan(ctx, key, q[:, P:], k[:, P:], v[:, P:], g[:, P:], state, state, o[:, P:], T - P, T, chunk)
    torch.cuda.synchronize()
    assert bits_equal(o, o_cold), "restore+continue differs from the cold run"
    assert bits_equal(state, s_cold)
    # determinism: the cold run twice gives the same bits
    o2, s2, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk)
    assert bits_equal(o2, o_cold) and bits_equal(s2, s_cold)


def test_misaligned_restore_is_within_tolerance(esc, ctx):
    # a boundary off the chunk grid introduces a chunk split the cold run never had:
    # tolerance-only against the oracle
    B, H, dk, dv, T, chunk, P = 1, 4, 128, 128, 512, 64, 256 + 37
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(14,), gate="slow")
    o_ref, s_ref = oracle.linattn_recurrence(*si.as_f32())
    dev_in = scan_dev_inputs(si)
    o_a, s_p, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, n=P)
    o_b, s_t, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, s0=s_p, t0=P)
    o = torch.cat([o_a, o_b], dim=1)
    assert err_o(o.cpu().numpy(), o_ref) <= TOL_O
    assert_state_close(s_t, s_ref)


def test_kv_only_restore_diverges(esc, ctx):
    # Table 8: dropping or staling the recurrent fold must be visible.  With the configured
    # gate the state is forgotten in ~10 tokens, so the check looks at the first suffix tokens.
    B, H, dk, dv, T, chunk, P = 1, 4, 128, 128, 256, 64, 128
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(15,))
    o_ref, _ = oracle.linattn_recurrence(*si.as_f32())
    dev_in = scan_dev_inputs(si)
    _, s_p, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, n=P)
    o_good, _, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, s0=s_p, t0=P)
    o_drop, _, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, s0=None, t0=P)            # fold dropped
    _, s_stale, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, n=P - 64)
    o_stale, _, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, s0=s_stale, t0=P)        # stale fold
    head = slice(0, 10)
    ref = o_ref[:, P:][:, head]
    assert err_o(o_good[:, head].cpu().numpy(), ref) <= TOL_O
    assert err_o(o_drop[:, head].cpu().numpy(), ref) > 10 * TOL_O
    assert err_o(o_stale[:, head].cpu().numpy(), ref) > 10 * TOL_O


def test_scan_argument_errors(esc, ctx):
    key = esc.shape_key_make(1, 2, 64, 64, esc.DTYPE_BF16, esc.DTYPE_F32, 64)
    t = torch.zeros(4096, dtype=torch.float32, device=DEV)
    with pytest.raises(esc.EscError) as e:      # chunk differs from the key's
        esc.linattn_scan(ctx, key, t, t, t, t, None, t, t, 1, 1, 128)
    assert e.value.code == esc.ERR_MISMATCH
    with pytest.raises(esc.EscError) as e:      # misaligned q
        esc.linattn_scan(ctx, key, t.data_ptr() + 2, t, t, t, None, t, t, 1, 1, 64)
    assert e.value.code == esc.ERR_UNALIGNED
    with pytest.raises(esc.EscError) as e:      # t_stride < T
        esc.linattn_scan(ctx, key, t, t, t, t, None, t, t, 8, 4, 64)
    assert e.value.code == esc.ERR_INVALID
    with pytest.raises(esc.EscError) as e:      # not a key
        esc.linattn_scan(ctx, 12345, t, t, t, t, None, t, t, 1, 1, 64)
    assert e.value.code == esc.ERR_INVALID


def _check_sampled_heads(si, o, s, pairs, t_from=0):
    """oracle over the whole sequence for each sampled (b, h); compares o[:, t_from:] and the final state."""
    q, k, v, g = si.as_f32()
    for (b, h) in pairs:
        sl = (slice(b, b + 1), slice(None), slice(h, h + 1))
        o_ref, s_ref = oracle.linattn_recurrence(q[sl], k[sl], v[sl], g[sl])
        eo = err_o(o[b:b + 1, :, h:h + 1].cpu().numpy(), o_ref[:, t_from:])
        assert eo <= TOL_O, "o error %.3e at (b, h) = %s" % (eo, (b, h))
        assert_state_close(s[b:b + 1, h:h + 1], s_ref, "at (b, h) = %s" % ((b, h),))


def test_full_size_config2_sampled(esc, ctx):
    # BASELINE config 2's cold scan at full size (B1 H16 d128, T = 16384 + 64, chunk 64) in the launch
    # configuration bench.py times; the oracle checks a seeded sample of heads over the whole sequence.
    B, H, dk, dv, T, chunk = 1, 16, 128, 128, 16384 + 64, 64
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(16,))
    o, s, _ = run_scan(esc, ctx, scan_dev_inputs(si), B, T, H, dk, dv, chunk)
    _check_sampled_heads(si, o, s, sample_heads(B, H, 3, 16))


@pytest.mark.parametrize("B,T,chunk", [
    (4, 2048, 64),      # 64 (b,h) scans: several waves of CTAs on 148 SMs
    (2, 8192, 128),
    (4, 8192, 64),      # the B = 4 tile at a length bench.py times
    (1, 32768, 64),
    (1, 65536, 64),     # 1024 chunks: every barrier parity wraps 256+ times, the gate warp batches 256 times
    (4, 32768, 64),     # the largest B x T bench.py's sweep times
])
def test_config4_sweep_points_sampled(esc, ctx, B, T, chunk):
    # BASELINE config 4 (scan sweep: B 1-4, H16, d128, T 2k-64k, chunk 64/128) at full head shape, every (B, T) the
    # bench's scan_sweep publishes a number for that the three historical points did not cover: the oracle checks a
    # seeded sample of (b, h) scans over the whole sequence; a chunk-aligned boundary at T/2 must continue bit-identically
    # to the cold run, a misaligned one (T/2 + 37) within tolerance.
    H, dk, dv = 16, 128, 128
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(17, B, T, chunk))
    dev_in = scan_dev_inputs(si)
    o_cold, s_cold, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk)
    pairs = sample_heads(B, H, 3, 17, B, T, chunk)
    _check_sampled_heads(si, o_cold, s_cold, pairs)
    P = (T // 2) // chunk * chunk
    _, s_p, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, n=P)
    o_b, s_t, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, s0=s_p, t0=P)
    assert bits_equal(o_b, o_cold[:, P:]) and bits_equal(s_t, s_cold)
    del o_b, s_t
    Pm = P + 37
    _, s_pm, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, n=Pm)
    o_m, s_tm, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, s0=s_pm, t0=Pm)
    _check_sampled_heads(si, o_m, s_tm, pairs[:1], t_from=Pm)   # misaligned restore: oracle tolerance only


@pytest.mark.parametrize("B", [1, 2, 4])
def test_back_to_back_scans_on_one_stream_are_ordered(esc, ctx, B):
    # the scan kernel allows programmatic dependent launch: a following scan may start its on-chip setup early but must
    # not read the state the previous one is still writing.  20 chained in-place suffix scans == one scan over all tokens
    # (B = 1: the 16-column tile; B = 2, 4: the 32-column tile).
    H, dk, dv, chunk, n, T = 16, 128, 128, 64, 20, 20 * 64
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(18,), gate="slow")
    dev_in = scan_dev_inputs(si)
    o_cold, s_cold, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk)
    key = esc.shape_key_make(B, H, dk, dv, esc.DTYPE_BF16, esc.DTYPE_F32, chunk)
    q, k, v, g = dev_in
    state = torch.zeros((B, H, dk, dv), dtype=torch.float32, device=DEV)
    o = torch.zeros((B, T, H, dv), dtype=torch.float32, device=DEV)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    for rep in range(3):
        state.zero_()
        stream.wait_stream(torch.cuda.current_stream())
        for i in range(n):
            t0 = i * 64
            esc.linattn_scan(ctx, key, q[:, t0:], k[:, t0:], v[:, t0:], g[:, t0:], state, state, o[:, t0:], 64, T, chunk,
                             stream=stream)
        stream.synchronize()
        assert bits_equal(o, o_cold) and bits_equal(state, s_cold)


def test_tile_is_a_function_of_the_key_not_of_T(esc, ctx):
    # DESIGN.md reading 11 / 26: the d_v tile is chosen from (B, H, d_v) and the device only; the call never sees T
    k1 = esc.shape_key_make(1, 16, 128, 128, esc.DTYPE_BF16, esc.DTYPE_F32, 64)
    k2 = esc.shape_key_make(2, 16, 128, 128, esc.DTYPE_BF16, esc.DTYPE_F32, 64)
    k4 = esc.shape_key_make(4, 16, 128, 128, esc.DTYPE_BF16, esc.DTYPE_BF16, 128)
    ks = esc.shape_key_make(1, 2, 64, 64, esc.DTYPE_BF16, esc.DTYPE_F32, 64)
    assert esc.scan_tile_columns(ctx, k1) == 16 and esc.scan_tile_columns(ctx, ks) == 16     # one wave of 16-column CTAs
    assert esc.scan_tile_columns(ctx, k2) == 32 and esc.scan_tile_columns(ctx, k4) == 32


@pytest.mark.parametrize("B,H,dk,dv,out_bf16", [
    (2, 16, 128, 128, False),    # 32-column tile (the historical case)
    (1, 16, 128, 128, False),    # 16-column tile
    (4, 16, 128, 128, True),     # 32-column tile, bf16 o
    (2, 20, 64, 64, False),      # d = 64, 32-column tile, clusters of 2
    (1, 4, 64, 64, True),        # d = 64, 16-column tile, bf16 o
])
def test_short_call_variant_matches_long_call_prefix_bitwise(esc, ctx, B, H, dk, dv, out_bf16):
    # calls of up to 128 tokens launch the kernel without its cluster (whole-tile TMA loads instead of multicast row slices);
    # the arithmetic is the same.  Causality makes o[:, :T] of a long call a function of the first T tokens only, so it must
    # equal the short call's o bit for bit, ragged T included; so must the carried state at chunk multiples.  Every d_v tile,
    # d = 64 and the bf16-o variant are covered (the proof is by test, reading 26).
    chunk, T_long = 64, 448
    si = synth.scan_inputs(B, T_long, H, dk, dv, seed_ids=(21, B, H, dk), gate="slow")
    s0 = synth.scan_state(B, H, dk, dv, seed_ids=(21,), scale=0.3)
    dev_in = scan_dev_inputs(si)
    s0_dev = torch.from_numpy(s0).to(DEV)
    o_long, _, _ = run_scan(esc, ctx, dev_in, B, T_long, H, dk, dv, chunk, s0=s0_dev, out_bf16=out_bf16)
    for T in (1, 37, 64, 100, 128):
        o_short, s_short, _ = run_scan(esc, ctx, dev_in, B, T_long, H, dk, dv, chunk, s0=s0_dev, n=T, out_bf16=out_bf16)
        assert bits_equal(o_short[:, :T], o_long[:, :T]), T
        if T % chunk == 0:   # continue the long way from the short call's state: the rest of the long run, bit for bit
            o_rest, _, _ = run_scan(esc, ctx, dev_in, B, T_long, H, dk, dv, chunk, s0=s_short, t0=T, out_bf16=out_bf16)
            assert bits_equal(o_rest, o_long[:, T:]), T


def test_seeded_shape_fuzz_vs_oracle(esc, ctx):
    # 24 seeded random (B, H, d_k, d_v, T, chunk, gate, S_0) combinations, ragged T included: every one within the gates,
    # every chunk-aligned restore bit-identical to its cold run
    rng = np.random.default_rng(20537)
    for it in range(24):
        B, H = int(rng.integers(1, 4)), int(rng.integers(1, 6))
        dk, dv = int(rng.choice([64, 128])), int(rng.choice([64, 128]))
        chunk = int(rng.choice([64, 128]))
        T = int(rng.integers(1, 420))
        gate = str(rng.choice(["fast", "slow", "one"]))
        si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(19, it), gate=gate)
        s0 = synth.scan_state(B, H, dk, dv, seed_ids=(19, it), scale=0.3) if it % 2 else None
        dev_in = scan_dev_inputs(si)
        o, s, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, s0=None if s0 is None else to_dev(s0))
        o_ref, s_ref = oracle.linattn_recurrence(*si.as_f32(), None if s0 is None else s0.astype(np.float64))
        tag = (it, B, H, dk, dv, T, chunk, gate)
        assert err_o(o.cpu().numpy(), o_ref) <= TOL_O, tag
        assert_state_close(s, s_ref, str(tag))
        P = (T // 2) // chunk * chunk
        if P > 0:
            _, s_p, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, s0=None if s0 is None else to_dev(s0), n=P)
            o_b, s_t, _ = run_scan(esc, ctx, dev_in, B, T, H, dk, dv, chunk, s0=s_p, t0=P)
            assert bits_equal(o_b, o[:, P:]) and bits_equal(s_t, s), tag
