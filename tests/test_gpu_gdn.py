"""-m gpu parity of esc_gdn_scan (gated delta rule) and esc_causal_conv (convolution state) through the C ABI against
oracle/gdn_oracle.c (reading 25).  Same bars as the linear-attention scan: o within 2e-3
(inf-norm ratio), S within 1e-3 (relative Frobenius); restore + continue bit-identical to the cold run at every boundary
that is a multiple of the kernel's (= the key's) 64-token chunk, within the gates elsewhere."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_20537_b200 import synth
from gpu_util import DEV, TOL_O, TOL_S, assert_state_close, bits_equal, err_o, err_s, esc_mod, sample_heads, scan_dev_inputs, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def esc():
    return esc_mod()


@pytest.fixture(scope="module")
def ctx(esc):
    c = esc.Ctx(0)
    yield c
    c.close()


def run_gdn(esc, ctx, dev_in, beta, B, T, H, dk, dv, s0=None, t0=0, n=None):
    q, k, v, g = dev_in
    t_stride = q.shape[1]
    n = T - t0 if n is None else n
    key = esc.shape_key_make(B, H, dk, dv, esc.DTYPE_BF16, esc.DTYPE_F32, 64)
    o = torch.full((B, t_stride, H, dv), float("nan"), dtype=torch.float32, device=DEV)
    s_out = torch.full((B, H, dk, dv), float("nan"), dtype=torch.float32, device=DEV)
    esc.gdn_scan(ctx, key, q[:, t0:], k[:, t0:], v[:, t0:], g[:, t0:], beta[:, t0:], s0, s_out, o[:, t0:], n, t_stride)
    torch.cuda.synchronize()
    return o[:, t0:t0 + n], s_out, o


@pytest.mark.parametrize("B,H,dk,dv,T,gate", [
    (1, 2, 64, 64, 256, "fast"),
    (2, 3, 128, 128, 300, "fast"),       # ragged: 300 = 4 chunks + 44
    (1, 16, 128, 128, 512, "slow"),      # config-1 head shape, slow decay: the carried state matters throughout
    (1, 2, 128, 64, 1, "fast"),
    (1, 1, 64, 128, 65, "one"),
])
@pytest.mark.parametrize("with_s0", [False, True])
def test_gdn_vs_oracle(esc, ctx, B, H, dk, dv, T, gate, with_s0):
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(70, T, H), gate=gate)
    beta = synth.gdn_beta(B, T, H, seed_ids=(70, T, H))
    s0 = synth.scan_state(B, H, dk, dv, seed_ids=(71,), scale=0.3) if with_s0 else None
    o, s, o_full = run_gdn(esc, ctx, scan_dev_inputs(si), to_dev(beta), B, T, H, dk, dv, s0=None if s0 is None else to_dev(s0))
    q, k, v, g = si.as_f32()
    o_ref, s_ref = oracle.gdn_recurrence(q, k, v, g, beta, None if s0 is None else s0.astype(np.float64))
    assert err_o(o.cpu().numpy(), o_ref) <= TOL_O
    assert_state_close(s, s_ref)
    assert err_o(o.cpu().numpy(), o_ref) <= 5e-5 and err_s(s.cpu().numpy(), s_ref) <= 5e-5   # two-term bf16 operands, fp32 accumulation: far inside the gates


@pytest.mark.parametrize("T", [128, 191, 192, 257, 320, 449, 512, 577, 1100])
@pytest.mark.parametrize("dv", [64, 128])
def test_gdn_chunk_counts_around_the_cluster_period(esc, ctx, T, dv):
    """The chunk inverses are computed by the CTAs of a cluster in turn (chunk c by CTA c % 4) and pushed to the others two
    operand slots deep: chunk counts of 2 ... 18 cover every phase of that rotation, ragged tails included; d_v = 64 is one
    cluster per head, d_v = 128 two."""
    B, H, dk = 1, 2, 128
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(75, T, dv), gate="slow")
    beta = synth.gdn_beta(B, T, H, seed_ids=(75, T, dv))
    s0 = synth.scan_state(B, H, dk, dv, seed_ids=(76,), scale=0.3)
    o, s, _ = run_gdn(esc, ctx, scan_dev_inputs(si), to_dev(beta), B, T, H, dk, dv, s0=to_dev(s0))
    q, k, v, g = si.as_f32()
    o_ref, s_ref = oracle.gdn_recurrence(q, k, v, g, beta, s0.astype(np.float64))
    assert err_o(o.cpu().numpy(), o_ref) <= 5e-5 and err_s(s.cpu().numpy(), s_ref) <= 5e-5
    assert_state_close(s, s_ref)
    # and the same call twice gives the same bits (no dependence on the arrival order of the pushed inverses)
    o2, s2, _ = run_gdn(esc, ctx, scan_dev_inputs(si), to_dev(beta), B, T, H, dk, dv, s0=to_dev(s0))
    assert bits_equal(o, o2) and bits_equal(s, s2)


@pytest.mark.parametrize("dk,dv", [(128, 128), (64, 64)])
def test_gdn_short_call_matches_long_call_prefix_bitwise(esc, ctx, dk, dv):
    """Calls of up to 64 tokens launch without the cluster (every CTA inverts its own chunk); longer calls share the inverses
    across four d_v slices.  Same instructions on the same inputs: the first 64 tokens of a long call and a 64-token call give the
    same o bits, and a chain of 64-token calls ends in the long call's state."""
    B, H, T = 1, 3, 256
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(77, dk), gate="slow")
    beta = to_dev(synth.gdn_beta(B, T, H, seed_ids=(77, dk)))
    s0 = to_dev(synth.scan_state(B, H, dk, dv, seed_ids=(78,), scale=0.3))
    dev_in = scan_dev_inputs(si)
    o_long, s_long, _ = run_gdn(esc, ctx, dev_in, beta, B, T, H, dk, dv, s0=s0)
    s = s0
    for t0 in range(0, T, 64):
        o_b, s, _ = run_gdn(esc, ctx, dev_in, beta, B, T, H, dk, dv, s0=s, t0=t0, n=64)
        assert bits_equal(o_b, o_long[:, t0:t0 + 64]), t0
    assert bits_equal(s, s_long)


def test_gdn_restore_continue_bit_identical_at_chunk_boundaries(esc, ctx):
    B, H, dk, dv, T = 1, 4, 128, 128, 333
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(72,), gate="slow")
    beta = to_dev(synth.gdn_beta(B, T, H, seed_ids=(72,)))
    dev_in = scan_dev_inputs(si)
    o_cold, s_cold, _ = run_gdn(esc, ctx, dev_in, beta, B, T, H, dk, dv)
    for P in (64, 128, 192, 256, 320):       # chunk-aligned (64) boundaries, on and off the 256-token gate-batch grid
        _, s_p, _ = run_gdn(esc, ctx, dev_in, beta, B, T, H, dk, dv, n=P)
        o_b, s_t, _ = run_gdn(esc, ctx, dev_in, beta, B, T, H, dk, dv, s0=s_p, t0=P)
        assert bits_equal(o_b, o_cold[:, P:]) and bits_equal(s_t, s_cold), P
    for P in (16, 304, 101, 332):            # misaligned: a different chunk grid, the same function to rounding
        _, s_p, _ = run_gdn(esc, ctx, dev_in, beta, B, T, H, dk, dv, n=P)
        o_b, s_t, _ = run_gdn(esc, ctx, dev_in, beta, B, T, H, dk, dv, s0=s_p, t0=P)
        assert err_o(o_b.cpu().numpy(), o_cold[:, P:].cpu().numpy().astype(np.float64)) <= 1e-4, P
        assert err_s(s_t.cpu().numpy(), s_cold.cpu().numpy().astype(np.float64)) <= 1e-4, P
    # through a capsule: fold state + convolution window as rows of one buffer set
    key = esc.shape_key_make(B, H, dk, dv, esc.DTYPE_BF16, esc.DTYPE_F32, 64)
    state = torch.zeros((B, H, dk, dv), dtype=torch.float32, device=DEV)
    conv_st = torch.randn((B, 256, 3), dtype=torch.float32, device=DEV)
    live = esc.bufset_create(ctx, [("L00.lin.state", state, state.numel() * 4, state.numel() * 4, 0, 1, 0),
                                   ("L00.lin.conv", conv_st, conv_st.numel() * 4, conv_st.numel() * 4, 0, 1, 0)])
    q, k, v, g = dev_in
    o = torch.zeros((B, T, H, dv), dtype=torch.float32, device=DEV)
    P = 128
    esc.gdn_scan(ctx, key, q, k, v, g, beta, None, state, o, P, T)
    slab = torch.empty(live.capsule_bytes(P)[0], dtype=torch.uint8, device=DEV)
    cap = esc.snapshot(live, P, 0, slab)
    keep_conv = conv_st.clone()
    state.fill_(float("nan"))
    conv_st.fill_(float("nan"))
    esc.restore(live, cap)
    esc.gdn_scan(ctx, key, q[:, P:], k[:, P:], v[:, P:], g[:, P:], beta[:, P:], state, state, o[:, P:], T - P, T)
    torch.cuda.synchronize()
    assert bits_equal(o, o_cold) and bits_equal(state, s_cold) and bits_equal(conv_st, keep_conv)


def test_gdn_full_size_sampled(esc, ctx):
    B, H, dk, dv, T = 1, 16, 128, 128, 4096 + 64
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(73,))
    beta = synth.gdn_beta(B, T, H, seed_ids=(73,))
    o, s, _ = run_gdn(esc, ctx, scan_dev_inputs(si), to_dev(beta), B, T, H, dk, dv)
    heads = sorted(h for _, h in sample_heads(B, H, 3, 73))
    q, k, v, g = si.as_f32()
    o_ref, s_ref = oracle.gdn_recurrence(q[:, :, heads], k[:, :, heads], v[:, :, heads], g[:, :, heads], beta[:, :, heads])
    assert err_o(o[:, :, heads].cpu().numpy(), o_ref) <= TOL_O
    assert_state_close(s[:, heads], s_ref)


def test_gdn_errors(esc, ctx):
    key_bf = esc.shape_key_make(1, 2, 64, 64, esc.DTYPE_BF16, esc.DTYPE_BF16, 64)
    x = torch.zeros(16, device=DEV)
    assert esc.lib.esc_gdn_scan(ctx.h, key_bf, *([x.data_ptr()] * 8), 1, 1, None) == esc.ERR_UNSUPPORTED
    key = esc.shape_key_make(1, 2, 64, 64, esc.DTYPE_BF16, esc.DTYPE_F32, 64)
    assert esc.lib.esc_gdn_scan(ctx.h, key, *([x.data_ptr()] * 5), None, None, x.data_ptr(), 1, 1, None) == esc.ERR_INVALID
    assert esc.lib.esc_gdn_scan(ctx.h, key, *([x.data_ptr() + 2] * 8), 1, 1, None) == esc.ERR_UNALIGNED


@pytest.mark.parametrize("B,T,C,W,silu", [(2, 300, 64, 4, False), (1, 1000, 256, 4, True), (1, 2, 8, 4, False), (3, 17, 24, 1, True),
                                          (1, 64, 6144, 4, True),
                                          # short calls take short runs (4 or 8 tokens per thread) and the first run writes the carried
                                          # window itself: every window size, T below / at / above W - 1, T not a multiple of a run
                                          (1, 7, 512, 8, True), (1, 8, 512, 8, False), (2, 9, 1024, 8, True), (1, 13, 2048, 5, False),
                                          (1, 3, 512, 4, True), (1, 4, 512, 4, False), (1, 67, 6144, 2, True), (2, 130, 6144, 7, True),
                                          # long calls: full 48-token runs (the per-thread cp.async ring wraps three times), a ragged
                                          # last run; the split at T // 2 takes 24-token runs
                                          (1, 2500, 6144, 4, True), (2, 1203, 6144, 3, False)])
def test_causal_conv_vs_oracle_and_continuation(esc, ctx, B, T, C, W, silu):
    x_bits, w, st = synth.conv_inputs(B, T, C, W, seed_ids=(80, T, C))
    x = to_dev(x_bits.view(np.int16)).view(torch.bfloat16)
    wd, s_in = to_dev(w), to_dev(st)
    # y sits between two canaries: a store outside [B, T, C] (a run or a ring slot past the ragged end) would show
    guard = 4096
    ybuf = torch.full((guard + B * T * C + guard,), -12345.0, dtype=torch.float32, device=DEV)
    y = ybuf[guard:guard + B * T * C].view(B, T, C)
    y.fill_(float("nan"))
    s_out = torch.full((B, C, max(W - 1, 1)), float("nan"), dtype=torch.float32, device=DEV)
    flags = esc.CONV_SILU if silu else 0
    esc.causal_conv(ctx, x, wd, s_in if W > 1 else None, s_out, y, B, T, T, C, W, flags)
    torch.cuda.synchronize()
    assert bool((ybuf[:guard] == -12345.0).all()) and bool((ybuf[guard + B * T * C:] == -12345.0).all())
    y_ref, s_ref = oracle.causal_conv(synth.bf16_bits_to_f32(x_bits), w, st.astype(np.float64) if W > 1 else None, silu=silu)
    assert np.abs(y.cpu().numpy() - y_ref).max() <= 1e-5 * max(1.0, np.abs(y_ref).max())
    if W > 1:
        assert np.array_equal(s_out.cpu().numpy()[:, :, :W - 1].astype(np.float64), s_ref)    # the window is a copy of inputs: exact
        # split at P with the carried window, in place (state_in == state_out): bit-identical to the single call
        for P in (1, T // 2):
            if P >= T:
                continue
            y2 = torch.full_like(y, float("nan"))
            s_io = s_in.clone()
            esc.causal_conv(ctx, x, wd, s_io, s_io, y2, B, P, T, C, W, flags)
            y2b = torch.full((B, T - P, C), float("nan"), dtype=torch.float32, device=DEV)
            esc.causal_conv(ctx, x[:, P:], wd, s_io, s_io, y2b, B, T - P, T, C, W, flags)
            torch.cuda.synchronize()
            # y is dense in T per call: the first call wrote [B, P, C] at the head of y2's storage
            y_first = y2.view(-1)[: B * P * C].view(B, P, C)
            assert bits_equal(torch.cat([y_first, y2b], dim=1), y) and bits_equal(s_io[:, :, :W - 1], s_out[:, :, :W - 1])
