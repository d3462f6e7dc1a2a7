"""Pins for the scan oracle (CPU only).  Each test checks oracle.linattn_recurrence against
something the mathematics fixes *other than itself*: the O(T^2) closed form by brute force,
library routines the definition reduces to in special cases, a hand-computed example,
invariants.  A dropped term, wrong sign/index or transposed operand fails at least one.

Definition pinned: north_star / SURVEY.md §8(c):  S_t = g_t S_{t-1} + k_t^T v_t,  o_t = q_t S_t.
"""
import numpy as np
import pytest
import scipy.signal

import oracle
from paper_2606_20537_b200 import synth


def _rand(B, T, H, dk, dv, seed, gate="fast"):
    si = synth.scan_inputs(B, T, H, dk, dv, seed_ids=(900, seed), gate=gate)
    return si.as_f32()


def closed_form(q, k, v, g, S0=None):
    """o_t = sum_{s<=t} (prod_{r=s+1..t} g_r) (q_t . k_s) v_s  +  (prod_{r=1..t} g_r) q_t S_0
    (BASELINE.json north_star's closed form + the S_0 term, reading #3), pure Python loops."""
    q, k, v, g = (np.asarray(a, np.float64) for a in (q, k, v, g))
    B, T, H, dk = q.shape
    dv = v.shape[-1]
    o = np.zeros((B, T, H, dv))
    for b in range(B):
        for h in range(H):
            for t in range(T):
                acc = np.zeros(dv)
                for s in range(t + 1):
                    w = 1.0
                    for r in range(s + 1, t + 1):
                        w *= g[b, r, h]
                    acc += w * float(np.dot(q[b, t, h], k[b, s, h])) * v[b, s, h]
                if S0 is not None:
                    w = 1.0
                    for r in range(t + 1):
                        w *= g[b, r, h]
                    acc += w * (q[b, t, h] @ np.asarray(S0[b, h], np.float64))
                o[b, t, h] = acc
    return o


def closed_form_state(k, v, g, S0=None):
    """S_T = sum_s (prod_{r=s+1..T} g_r) k_s^T v_s + (prod_r g_r) S_0."""
    k, v, g = (np.asarray(a, np.float64) for a in (k, v, g))
    B, T, H, dk = k.shape
    dv = v.shape[-1]
    S = np.zeros((B, H, dk, dv))
    for b in range(B):
        for h in range(H):
            for s in range(T):
                w = np.prod(g[b, s + 1:, h])
                S[b, h] += w * np.outer(k[b, s, h], v[b, s, h])
            if S0 is not None:
                S[b, h] += np.prod(g[b, :, h]) * np.asarray(S0[b, h], np.float64)
    return S


@pytest.mark.parametrize("B,T,H,dk,dv", [(1, 1, 1, 1, 1), (2, 17, 3, 3, 5), (1, 48, 2, 8, 4), (1, 64, 1, 2, 2)])
@pytest.mark.parametrize("with_s0", [False, True])
def test_closed_form_bruteforce(B, T, H, dk, dv, with_s0):
    q, k, v, g = _rand(B, T, H, dk, dv, seed=T * 7 + dk)
    S0 = synth.scan_state(B, H, dk, dv, seed_ids=(T,)).astype(np.float64) if with_s0 else None
    o, S = oracle.linattn_recurrence(q, k, v, g, S0)
    np.testing.assert_allclose(o, closed_form(q, k, v, g, S0), rtol=0, atol=1e-12)
    np.testing.assert_allclose(S, closed_form_state(k, v, g, S0), rtol=0, atol=1e-12)


def test_hand_example_T2_d1():
    # T = 2, d = 1, by hand:  S_1 = k1 v1 ; o_1 = q1 k1 v1 ; S_2 = g2 k1 v1 + k2 v2 ; o_2 = q2 S_2
    q = np.array([2.0, -3.0], np.float32).reshape(1, 2, 1, 1)
    k = np.array([0.5, 4.0], np.float32).reshape(1, 2, 1, 1)
    v = np.array([3.0, -1.0], np.float32).reshape(1, 2, 1, 1)
    g = np.array([0.25, 0.5], np.float32).reshape(1, 2, 1)
    o, S = oracle.linattn_recurrence(q, k, v, g)
    assert o.reshape(-1).tolist() == [2.0 * 0.5 * 3.0, -3.0 * (0.5 * 0.5 * 3.0 + 4.0 * -1.0)]  # [3.0, 9.75]
    assert S.reshape(-1).tolist() == [0.5 * 1.5 - 4.0]                                          # [-3.25]
    # with S_0 = 8:  S_1 = 0.25*8 + 1.5 = 3.5 ; S_2 = 0.5*3.5 - 4 = -2.25
    o, S = oracle.linattn_recurrence(q, k, v, g, np.full((1, 1, 1, 1), 8.0))
    assert o.reshape(-1).tolist() == [7.0, 6.75] and S.reshape(-1).tolist() == [-2.25]


def test_gate_one_reduces_to_masked_matmul():
    # g == 1:  o = tril(Q K^T) V ,  S_T = K^T V  (plain linear attention; numpy matmul)
    B, T, H, dk, dv = 2, 40, 2, 6, 5
    q, k, v, g = _rand(B, T, H, dk, dv, seed=1, gate="one")
    assert np.all(g == 1.0)
    o, S = oracle.linattn_recurrence(q, k, v, g)
    q64, k64, v64 = (a.astype(np.float64) for a in (q, k, v))
    for b in range(B):
        for h in range(H):
            A = np.tril(q64[b, :, h] @ k64[b, :, h].T)
            np.testing.assert_allclose(o[b, :, h], A @ v64[b, :, h], rtol=0, atol=1e-12)
            np.testing.assert_allclose(S[b, h], k64[b, :, h].T @ v64[b, :, h], rtol=0, atol=1e-12)


def test_scalar_constant_gate_is_first_order_iir():
    # dk = dv = 1, g == gamma:  S_t = gamma S_{t-1} + k_t v_t  is lfilter([1],[1,-gamma], k*v)
    T, gamma = 200, np.float32(0.9)
    q, k, v, _ = _rand(1, T, 1, 1, 1, seed=2)
    g = np.full((1, T, 1), gamma, np.float32)
    o, S = oracle.linattn_recurrence(q, k, v, g)
    x = (k.astype(np.float64) * v.astype(np.float64)).reshape(T)
    s_ref = scipy.signal.lfilter([1.0], [1.0, -float(gamma)], x)
    np.testing.assert_allclose(o.reshape(T), q.astype(np.float64).reshape(T) * s_ref, rtol=0, atol=1e-12)
    np.testing.assert_allclose(S.reshape(()), s_ref[-1], rtol=0, atol=1e-12)


def test_tiny_gate_forgets_everything():
    # g -> tiny:  o_t -> (q_t . k_t) v_t
    B, T, H, dk, dv = 1, 12, 2, 4, 3
    q, k, v, _ = _rand(B, T, H, dk, dv, seed=3)
    g = np.full((B, T, H), 1e-30, np.float32)
    o, _ = oracle.linattn_recurrence(q, k, v, g)
    ref = np.einsum("bthk,bthk->bth", q.astype(np.float64), k.astype(np.float64))[..., None] * v.astype(np.float64)
    np.testing.assert_allclose(o, ref, rtol=0, atol=1e-25)


def test_state_only_decay():
    # k = v = 0, S_0 != 0:  S_T = (prod g) S_0 ;  o_t = (prod_{r<=t} g_r) q_t S_0
    B, T, H, dk, dv = 2, 9, 2, 3, 4
    q, _, _, g = _rand(B, T, H, dk, dv, seed=4)
    z_k = np.zeros((B, T, H, dk), np.float32)
    z_v = np.zeros((B, T, H, dv), np.float32)
    S0 = synth.scan_state(B, H, dk, dv, seed_ids=(5,)).astype(np.float64)
    o, S = oracle.linattn_recurrence(q, z_k, z_v, g, S0)
    cum = np.cumprod(g.astype(np.float64), axis=1)
    np.testing.assert_allclose(S, cum[:, -1][:, :, None, None] * S0, rtol=1e-14)
    ref = cum[..., None] * np.einsum("bthk,bhkv->bthv", q.astype(np.float64), S0)
    np.testing.assert_allclose(o, ref, rtol=1e-13, atol=1e-15)


def test_linearity_in_v_and_state():
    B, T, H, dk, dv = 1, 20, 2, 4, 4
    q, k, v1, g = _rand(B, T, H, dk, dv, seed=6)
    _, _, v2, _ = _rand(B, T, H, dk, dv, seed=7)
    Sa = synth.scan_state(B, H, dk, dv, seed_ids=(8,)).astype(np.float64)
    Sb = synth.scan_state(B, H, dk, dv, seed_ids=(9,)).astype(np.float64)
    o1, S1 = oracle.linattn_recurrence(q, k, v1, g, Sa)
    o2, S2 = oracle.linattn_recurrence(q, k, v2, g, Sb)
    # exact fp32 sums are not generally representable: feed the sum as fp32 of (v1 + v2)/2 * 2 -> use scaling by 2 (exact)
    o3, S3 = oracle.linattn_recurrence(q, k, (2 * v1).astype(np.float32), g, 2 * Sa)
    np.testing.assert_allclose(o3, 2 * o1, rtol=0, atol=0)   # scaling by a power of two is exact
    np.testing.assert_allclose(S3, 2 * S1, rtol=0, atol=0)
    vs = (v1.astype(np.float64) + v2.astype(np.float64)).astype(np.float32)
    exact = np.array_equal(vs.astype(np.float64), v1.astype(np.float64) + v2.astype(np.float64))
    o4, S4 = oracle.linattn_recurrence(q, k, vs, g, Sa + Sb)
    tol = 1e-12 if exact else 1e-6
    np.testing.assert_allclose(o4, o1 + o2, rtol=0, atol=tol)
    np.testing.assert_allclose(S4, S1 + S2, rtol=0, atol=tol)


@pytest.mark.parametrize("P", [0, 1, 37, 64, 99, 100])
def test_restore_continue_is_bitwise_cold(P):
    # the sequential recurrence has no chunking: cold(0->T) == cold(0->P) ; continue(P->T from S_P), bit for bit
    B, T, H, dk, dv = 2, 100, 3, 8, 8
    q, k, v, g = _rand(B, T, H, dk, dv, seed=10)
    o_cold, S_cold = oracle.linattn_recurrence(q, k, v, g)
    o_a, S_P = oracle.linattn_recurrence(q[:, :P], k[:, :P], v[:, :P], g[:, :P]) if P else (np.zeros((B, 0, H, dv)), None)
    o_b, S_T = oracle.linattn_recurrence(q[:, P:], k[:, P:], v[:, P:], g[:, P:], S_P)
    assert np.array_equal(np.concatenate([o_a, o_b], axis=1).view(np.uint64), o_cold.view(np.uint64))
    assert np.array_equal(S_T.view(np.uint64), S_cold.view(np.uint64))


def test_c_oracle_matches_numpy_twin():
    for (B, T, H, dk, dv, gate) in [(2, 33, 3, 5, 7, "fast"), (1, 130, 2, 16, 16, "slow"), (1, 64, 2, 64, 64, "fast")]:
        q, k, v, g = _rand(B, T, H, dk, dv, seed=T, gate=gate)
        S0 = synth.scan_state(B, H, dk, dv, seed_ids=(T,)).astype(np.float64)
        o_c, S_c = oracle.linattn_recurrence(q, k, v, g, S0)
        o_n, S_n = oracle.linattn_recurrence_np(q, k, v, g, S0)
        np.testing.assert_allclose(o_c, o_n, rtol=0, atol=1e-12)
        np.testing.assert_allclose(S_c, S_n, rtol=0, atol=1e-12)


def test_t_stride_and_thread_count_do_not_change_bits():
    B, Tbuf, T, H, dk, dv = 2, 50, 31, 2, 4, 4
    q, k, v, g = _rand(B, Tbuf, H, dk, dv, seed=11)
    o1, S1 = oracle.linattn_recurrence(q, k, v, g, T=T, n_threads=1)
    o2, S2 = oracle.linattn_recurrence(q[:, :T], k[:, :T], v[:, :T], g[:, :T], n_threads=4)
    assert np.array_equal(o1.view(np.uint64), o2.view(np.uint64)) and np.array_equal(S1.view(np.uint64), S2.view(np.uint64))


def test_empty_T():
    q, k, v, g = _rand(1, 4, 2, 4, 4, seed=12)
    S0 = synth.scan_state(1, 2, 4, 4, seed_ids=(13,)).astype(np.float64)
    o, S = oracle.linattn_recurrence(q, k, v, g, S0, T=0)
    assert o.shape == (1, 0, 2, 4) and np.array_equal(S, S0)


# ---------------------------------------------------------------------------------------
# the chunk algebra the CUDA kernel implements, evaluated in fp64 numpy,
# must equal the sequential definition — validates the derivation before any CUDA.
#   o_i    = exp(b_i) q_i S_prev + sum_{j<=i} exp(b_i - b_j) (q_i . k_j) v_j
#   S_next = exp(b_C) S_prev + sum_i exp(b_C - b_i) k_i^T v_i ,   b_i = sum_{r<=i} ln g_r
# ---------------------------------------------------------------------------------------
def chunked_fp64(q, k, v, g, S0, C):
    q, k, v, g = (np.asarray(a, np.float64) for a in (q, k, v, g))
    B, T, H, dk = q.shape
    dv = v.shape[-1]
    S = np.zeros((B, H, dk, dv)) if S0 is None else np.array(S0, np.float64)
    o = np.zeros((B, T, H, dv))
    for c0 in range(0, T, C):
        c1 = min(T, c0 + C)
        n = c1 - c0
        for b in range(B):
            for h in range(H):
                bb = np.cumsum(np.log(g[b, c0:c1, h]))
                Q, K, V = q[b, c0:c1, h], k[b, c0:c1, h], v[b, c0:c1, h]
                D = np.where(np.tril(np.ones((n, n), bool)), np.exp(np.minimum(bb[:, None] - bb[None, :], 0.0)), 0.0)
                o[b, c0:c1, h] = ((Q @ K.T) * D) @ V + np.exp(bb)[:, None] * (Q @ S[b, h])
                S[b, h] = np.exp(bb[-1]) * S[b, h] + K.T @ (V * np.exp(bb[-1] - bb)[:, None])
    return o, S


@pytest.mark.parametrize("C", [1, 7, 64, 128])
@pytest.mark.parametrize("gate", ["fast", "slow"])
def test_chunk_algebra_equals_definition(C, gate):
    B, T, H, dk, dv = 1, 203, 2, 16, 12   # T not a multiple of any C > 1 used
    q, k, v, g = _rand(B, T, H, dk, dv, seed=14, gate=gate)
    S0 = synth.scan_state(B, H, dk, dv, seed_ids=(15,)).astype(np.float64)
    o_ref, S_ref = oracle.linattn_recurrence(q, k, v, g, S0)
    o, S = chunked_fp64(q, k, v, g, S0, C)
    np.testing.assert_allclose(o, o_ref, rtol=0, atol=1e-11)
    np.testing.assert_allclose(S, S_ref, rtol=0, atol=1e-11)


def test_synth_inputs_are_as_specified():
    si = synth.scan_inputs(1, 256, 2, 64, 64, seed_ids=(0, 0), gate="fast")
    q, k, v, g = si.as_f32()
    # L2-normalised (up to bf16 rounding), gate in (0,1], mean ~0.5; same seed -> same bits
    assert np.allclose(np.linalg.norm(q.astype(np.float64), axis=-1), 1.0, atol=5e-3)
    assert np.allclose(np.linalg.norm(k.astype(np.float64), axis=-1), 1.0, atol=5e-3)
    assert g.dtype == np.float32 and np.all(g > 0) and np.all(g <= 1) and abs(g.mean() - 0.5) < 0.05
    si2 = synth.scan_inputs(1, 256, 2, 64, 64, seed_ids=(0, 0), gate="fast")
    assert np.array_equal(si.q_bits, si2.q_bits) and np.array_equal(si.g, si2.g)
    # bf16 round trip is exact on already-rounded values and RNE on a known tie
    assert np.array_equal(synth.f32_to_bf16_bits(q), si.q_bits)
    tie = np.array([1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8], np.float32)   # ties -> even mantissa
    assert synth.bf16_bits_to_f32(synth.f32_to_bf16_bits(tie)).tolist() == [1.0, 1.0 + 2.0 ** -6]
    assert np.array_equal(oracle.bf16_bits_to_f32(si.v_bits), v)
