"""Pins of the gated-delta-rule and causal-convolution oracles (oracle/gdn_oracle.c) against things other than themselves:
closed forms, the delta rule's overwrite property, the already-pinned gated linear-attention oracle on orthogonal keys,
an affine-map restatement with numpy matmul, scipy.signal.lfilter, and the restore-continue invariant."""
import numpy as np
import pytest
import scipy.signal

import oracle


def _rand(B, T, H, dk, dv, seed, orth=False):
    r = np.random.default_rng([20537, 9, seed])
    q = r.standard_normal((B, T, H, dk)).astype(np.float32)
    k = r.standard_normal((B, T, H, dk))
    if orth:                                   # mutually orthonormal keys per (b, h): needs T <= dk
        assert T <= dk
        for b in range(B):
            for h in range(H):
                Q, _ = np.linalg.qr(r.standard_normal((dk, T)))
                k[b, :, h] = Q.T
    else:
        k /= np.linalg.norm(k, axis=-1, keepdims=True)
    v = r.standard_normal((B, T, H, dv)).astype(np.float32)
    g = (1.0 / (1.0 + np.exp(r.standard_normal((B, T, H))))).astype(np.float32)
    beta = (1.0 / (1.0 + np.exp(-r.standard_normal((B, T, H))))).astype(np.float32)
    return q, k.astype(np.float32), v, g, beta


def test_hand_example_T1_T2():
    q = np.array([[[[2.0]], [[3.0]]]], np.float32)        # B=1, T=2, H=1, dk=dv=1
    k = np.array([[[[0.5]], [[1.0]]]], np.float32)
    v = np.array([[[[4.0]], [[-1.0]]]], np.float32)
    g = np.array([[[0.5], [0.25]]], np.float32)
    b = np.array([[[1.0], [0.5]]], np.float32)
    s0 = np.array([[[[8.0]]]])
    o, s = oracle.gdn_recurrence(q, k, v, g, b, s0)
    s1 = 0.5 * 8 + 1.0 * 0.5 * (4.0 - 0.5 * (0.5 * 8))      # = 4 + 0.5 * 2 = 5
    s2 = 0.25 * s1 + 0.5 * 1.0 * (-1.0 - 1.0 * 0.25 * s1)   # = 1.25 + 0.5 * (-2.25) = 0.125
    assert s1 == 5.0 and s2 == 0.125
    assert o[0, 0, 0, 0] == 2.0 * s1 and o[0, 1, 0, 0] == 3.0 * s2 and s[0, 0, 0, 0] == s2


def test_beta_zero_is_pure_decay():
    q, k, v, g, beta = _rand(2, 9, 2, 4, 3, 1)
    s0 = np.random.default_rng(3).standard_normal((2, 2, 4, 3))
    o, s = oracle.gdn_recurrence(q, k, v, g, np.zeros_like(beta), s0)
    cum = np.cumprod(g.astype(np.float64), axis=1)
    np.testing.assert_allclose(s, cum[:, -1, :, None, None] * s0, rtol=1e-13)
    np.testing.assert_allclose(o, np.einsum("bthk,bhkv->bthv", q.astype(np.float64), s0) * cum[..., None], rtol=1e-12, atol=1e-14)


def test_orthogonal_keys_beta_one_is_gated_linear_attention():
    # with mutually orthogonal keys and S_0 = 0 the memory never holds anything for a new key: u_t = 0, and the delta
    # rule reduces to S_t = a_t S_{t-1} + k_t^T v_t — the (independently pinned) gated linear-attention oracle
    q, k, v, g, beta = _rand(1, 6, 2, 8, 5, 2, orth=True)
    o, s = oracle.gdn_recurrence(q, k, v, g, np.ones_like(beta))
    o_ref, s_ref = oracle.linattn_recurrence(q, k, v, g)
    np.testing.assert_allclose(o, o_ref, rtol=0, atol=1e-6)     # keys are orthogonal to fp32 rounding only
    np.testing.assert_allclose(s, s_ref, rtol=0, atol=1e-6)


def test_delta_rule_overwrites_an_association():
    # a = 1, beta = 1, unit key written twice with different values: the memory returns the LAST value for that key and
    # is untouched for an orthogonal key (the property the delta rule is named for)
    dk, dv = 4, 3
    e0, e1 = np.eye(dk, dtype=np.float32)[0], np.eye(dk, dtype=np.float32)[1]
    k = np.stack([e0, e1, e0])[None, :, None, :]
    v = np.array([[1, 2, 3], [4, 5, 6], [7, 8, 9]], np.float32)[None, :, None, :]
    ones = np.ones((1, 3, 1), np.float32)
    _, s = oracle.gdn_recurrence(k, k, v, ones, ones)
    np.testing.assert_array_equal(e0.astype(np.float64) @ s[0, 0], [7, 8, 9])
    np.testing.assert_array_equal(e1.astype(np.float64) @ s[0, 0], [4, 5, 6])


def test_affine_map_restatement_with_numpy_matmul():
    # S_t = A_t S_{t-1} + B_t with A_t = a_t (I - beta_t k_t^T k_t), B_t = beta_t k_t^T v_t, chained by numpy matmul
    q, k, v, g, beta = _rand(1, 12, 2, 6, 4, 4)
    s0 = np.random.default_rng(5).standard_normal((1, 2, 6, 4))
    o, s = oracle.gdn_recurrence(q, k, v, g, beta, s0)
    for h in range(2):
        S = s0[0, h].copy()
        for t in range(12):
            kt = k[0, t, h].astype(np.float64)[None, :]
            A = float(g[0, t, h]) * (np.eye(6) - float(beta[0, t, h]) * kt.T @ kt)
            S = A @ S + float(beta[0, t, h]) * kt.T @ v[0, t, h].astype(np.float64)[None, :]
            np.testing.assert_allclose(o[0, t, h], q[0, t, h].astype(np.float64) @ S, rtol=1e-11, atol=1e-13)
        np.testing.assert_allclose(s[0, h], S, rtol=1e-11, atol=1e-13)


def test_restore_continue_invariant_bitwise():
    q, k, v, g, beta = _rand(2, 40, 2, 8, 8, 6)
    o, s = oracle.gdn_recurrence(q, k, v, g, beta)
    for P in (1, 17, 39):
        o1, s1 = oracle.gdn_recurrence(q, k, v, g, beta, T=P)
        o2, s2 = oracle.gdn_recurrence(q[:, P:], k[:, P:], v[:, P:], g[:, P:], beta[:, P:], s1)
        assert np.array_equal(np.concatenate([o1, o2], axis=1), o) and np.array_equal(s2, s)


@pytest.mark.parametrize("W", [1, 2, 4])
def test_causal_conv_is_an_fir_filter(W):
    r = np.random.default_rng([7, W])
    B, T, C = 2, 33, 5
    x = r.standard_normal((B, T, C)).astype(np.float32)
    w = r.standard_normal((C, W)).astype(np.float32)
    y, st = oracle.causal_conv(x, w)
    for b in range(B):
        for c in range(C):
            # tap i multiplies x_{t-W+1+i}: FIR coefficients are the taps reversed
            ref = scipy.signal.lfilter(w[c, ::-1].astype(np.float64), [1.0], x[b, :, c].astype(np.float64))
            np.testing.assert_allclose(y[b, :, c], ref, rtol=1e-12, atol=1e-14)
    if W > 1:
        np.testing.assert_array_equal(st, np.transpose(x[:, T - (W - 1):, :], (0, 2, 1)).astype(np.float64))
    # continuation with the carried window == one run, bitwise
    for P in (1, 2, 20):
        y1, s1 = oracle.causal_conv(x, w, T=P)
        y2, s2 = oracle.causal_conv(x[:, P:], w, s1)
        assert np.array_equal(np.concatenate([y1, y2], axis=1), y) and np.array_equal(s2, st)


def test_causal_conv_silu_branch_is_pinned():
    """The SiLU branch of the convolution oracle against things the mathematics fixes (not its own formula):
    the library logistic function scipy.special.expit, hand values, the odd-part identity silu(y) - silu(-y) = y,
    silu(0) = 0, the large-|y| limits, and the derivative at 0 (1/2) by a central difference."""
    # W = 1 with unit taps makes the pre-activation the input itself: y = x exactly, so known arguments can be fed in
    pts = np.array([0.0, 1.0, -1.0, 2.0, -2.0, 0.5, 30.0, -30.0, 1e-4, -1e-4], np.float32)
    x = pts[None, :, None]
    w = np.ones((1, 1), np.float32)
    y_lin, _ = oracle.causal_conv(x, w)
    np.testing.assert_array_equal(y_lin[0, :, 0], pts.astype(np.float64))
    ys, _ = oracle.causal_conv(x, w, silu=True)
    s = dict(zip(pts.tolist(), ys[0, :, 0].tolist()))
    # hand values: silu(1) = 1 / (1 + e^-1), silu(-1) = -1 / (1 + e), silu(2) = 2 / (1 + e^-2)
    assert s[0.0] == 0.0
    assert abs(s[1.0] - 0.7310585786300049) < 1e-15
    assert abs(s[-1.0] + 0.2689414213699951) < 1e-15
    assert abs(s[2.0] - 1.7615941559557649) < 1e-15
    # odd part: silu(y) - silu(-y) = y (sigmoid(y) + sigmoid(-y) = 1)
    for a in (1.0, 2.0, 30.0, float(np.float32(1e-4))):
        assert abs((s[a] - s[-a]) - a) < 1e-14 * max(1.0, a)
    # limits: silu(y) -> y for large y, -> 0- for very negative y
    assert abs(s[30.0] - 30.0) < 1e-11 and -1e-11 < s[-30.0] < 0.0
    # slope 1/2 at the origin
    h = float(np.float32(1e-4))
    assert abs((s[h] - s[-h]) / (2 * h) - 0.5) < 1e-12
    # against the library logistic function on a real convolution (W = 4, random taps and inputs)
    import scipy.special
    r = np.random.default_rng([7, 99])
    x = r.standard_normal((2, 33, 5)).astype(np.float32) * 3
    w = r.standard_normal((5, 4)).astype(np.float32)
    y, _ = oracle.causal_conv(x, w)
    ys, st = oracle.causal_conv(x, w, silu=True)
    np.testing.assert_allclose(ys, y * scipy.special.expit(y), rtol=1e-14, atol=1e-300)
    # the activation does not touch the carried window
    np.testing.assert_array_equal(st, oracle.causal_conv(x, w)[1])
