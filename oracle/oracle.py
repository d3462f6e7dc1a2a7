"""ctypes front-end of the C oracle + its numpy restatement.

ORACLE — TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  No code here is shared with,
imported by, or imports the CUDA path.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        path = _build.build()
        lib = C.CDLL(path)
        lib.esc_oracle_linattn.restype = C.c_int
        lib.esc_oracle_linattn.argtypes = [C.c_void_p] * 7 + [C.c_int64] * 6 + [C.c_int]
        lib.esc_oracle_gdn.restype = C.c_int
        lib.esc_oracle_gdn.argtypes = [C.c_void_p] * 8 + [C.c_int64] * 6 + [C.c_int]
        lib.esc_oracle_causal_conv.restype = C.c_int
        lib.esc_oracle_causal_conv.argtypes = [C.c_void_p] * 5 + [C.c_int64] * 5 + [C.c_int]
        lib.esc_oracle_max_threads.restype = C.c_int
        for name in ("esc_oracle_capsule_payload_bytes", "esc_oracle_capsule_slab_bytes"):
            f = getattr(lib, name)
            f.restype = C.c_int64
            f.argtypes = [C.c_void_p, C.c_int, C.c_uint64]
        lib.esc_oracle_capsule_seg_offset.restype = C.c_int64
        lib.esc_oracle_capsule_seg_offset.argtypes = [C.c_void_p, C.c_int, C.c_uint64, C.c_int, C.c_uint32]
        for name in ("esc_oracle_capsule_snapshot", "esc_oracle_capsule_restore"):
            f = getattr(lib, name)
            f.restype = C.c_int
            f.argtypes = [C.c_void_p, C.c_int, C.c_uint64, C.c_void_p, C.c_uint64]
        lib.esc_oracle_align_boundary.restype = C.c_uint64
        lib.esc_oracle_align_boundary.argtypes = [C.c_uint64, C.c_uint64]
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().esc_oracle_max_threads())


def bf16_bits_to_f32(bits: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns (uint16) to float32 (bf16 is the top half of fp32)."""
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32)


# --------------------------------------------------------------------------------------
# scan
# --------------------------------------------------------------------------------------
def linattn_recurrence(q, k, v, g, state_in=None, T=None, n_threads=0):
    """fp64 sequential recurrence (C).  north_star / SURVEY.md §8(c) "Definition".

    q, k: float32 [B, Tbuf, H, dk]; v: float32 [B, Tbuf, H, dv]; g: float32 [B, Tbuf, H]
    (fp32 containers holding the exact bf16 / fp32 input values); state_in: [B,H,dk,dv] or None.
    Only tokens [0, T) are consumed (T defaults to Tbuf).
    Returns (o float64 [B,T,H,dv], state_out float64 [B,H,dk,dv]).
    """
    q = np.ascontiguousarray(q, dtype=np.float32)
    k = np.ascontiguousarray(k, dtype=np.float32)
    v = np.ascontiguousarray(v, dtype=np.float32)
    g = np.ascontiguousarray(g, dtype=np.float32)
    B, Tbuf, H, dk = q.shape
    dv = v.shape[-1]
    if T is None:
        T = Tbuf
    assert k.shape == (B, Tbuf, H, dk) and v.shape == (B, Tbuf, H, dv) and g.shape == (B, Tbuf, H)
    assert 0 <= T <= Tbuf
    o = np.empty((B, T, H, dv), dtype=np.float64)
    s_out = np.empty((B, H, dk, dv), dtype=np.float64)
    s_in_p = None
    if state_in is not None:
        s_in = np.ascontiguousarray(state_in, dtype=np.float64)
        assert s_in.shape == (B, H, dk, dv)
        s_in_p = s_in.ctypes.data
    rc = _load().esc_oracle_linattn(q.ctypes.data, k.ctypes.data, v.ctypes.data, g.ctypes.data,
                                    s_in_p, o.ctypes.data, s_out.ctypes.data,
                                    B, T, Tbuf, H, dk, dv, int(n_threads))
    if rc != 0:
        raise RuntimeError("esc_oracle_linattn failed rc=%d" % rc)
    return o, s_out


def gdn_recurrence(q, k, v, g, beta, state_in=None, T=None, n_threads=0):
    """fp64 sequential gated delta rule (C; oracle/gdn_oracle.c, reading 25).  Shapes as linattn_recurrence,
    beta like g.  Returns (o float64 [B,T,H,dv], state_out float64 [B,H,dk,dv])."""
    q, k, v, g, beta = (np.ascontiguousarray(a, dtype=np.float32) for a in (q, k, v, g, beta))
    B, Tbuf, H, dk = q.shape
    dv = v.shape[-1]
    T = Tbuf if T is None else T
    assert k.shape == q.shape and v.shape == (B, Tbuf, H, dv) and g.shape == (B, Tbuf, H) == beta.shape and 0 <= T <= Tbuf
    o = np.empty((B, T, H, dv), dtype=np.float64)
    s_out = np.empty((B, H, dk, dv), dtype=np.float64)
    s_in_p = None
    if state_in is not None:
        s_in = np.ascontiguousarray(state_in, dtype=np.float64)
        assert s_in.shape == (B, H, dk, dv)
        s_in_p = s_in.ctypes.data
    rc = _load().esc_oracle_gdn(q.ctypes.data, k.ctypes.data, v.ctypes.data, g.ctypes.data, beta.ctypes.data, s_in_p,
                                o.ctypes.data, s_out.ctypes.data, B, T, Tbuf, H, dk, dv, int(n_threads))
    if rc != 0:
        raise RuntimeError("esc_oracle_gdn failed rc=%d" % rc)
    return o, s_out


def causal_conv(x, w, state_in=None, T=None, silu=False):
    """fp64 short causal depthwise convolution with carried window (C; oracle/gdn_oracle.c).
    x float32 [B,Tbuf,C]; w float32 [C,W]; state [B,C,W-1] (oldest first).  Returns (y [B,T,C], state_out [B,C,W-1])."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    w = np.ascontiguousarray(w, dtype=np.float32)
    B, Tbuf, Cc = x.shape
    W = w.shape[1]
    T = Tbuf if T is None else T
    assert w.shape[0] == Cc and 0 <= T <= Tbuf
    y = np.empty((B, T, Cc), dtype=np.float64)
    s_out = np.empty((B, Cc, max(W - 1, 0)), dtype=np.float64)
    s_in_p = None
    if state_in is not None:
        s_in = np.ascontiguousarray(state_in, dtype=np.float64)
        assert s_in.shape == (B, Cc, W - 1)
        s_in_p = s_in.ctypes.data
    rc = _load().esc_oracle_causal_conv(x.ctypes.data, w.ctypes.data, s_in_p, y.ctypes.data, s_out.ctypes.data,
                                        B, T, Tbuf, Cc, W, int(bool(silu)))
    if rc != 0:
        raise RuntimeError("esc_oracle_causal_conv failed rc=%d" % rc)
    return y, s_out


def linattn_recurrence_np(q, k, v, g, state_in=None):
    """The same definition restated in numpy (loop over t; vectorised over b,h only)."""
    q, k, v, g = (np.asarray(a, dtype=np.float64) for a in (q, k, v, g))
    B, T, H, dk = q.shape
    dv = v.shape[-1]
    S = np.zeros((B, H, dk, dv)) if state_in is None else np.array(state_in, dtype=np.float64)
    o = np.zeros((B, T, H, dv))
    for t in range(T):
        S = g[:, t, :, None, None] * S + k[:, t, :, :, None] * v[:, t, :, None, :]
        o[:, t] = np.einsum("bhk,bhkv->bhv", q[:, t], S)
    return o, S


# --------------------------------------------------------------------------------------
# capsule
# --------------------------------------------------------------------------------------
class _Row(C.Structure):
    _fields_ = [("base", C.c_void_p), ("capacity_bytes", C.c_uint64), ("fixed_bytes", C.c_uint64),
                ("bytes_per_token", C.c_uint64), ("n_seg", C.c_uint32), ("pad_", C.c_uint32),
                ("seg_stride", C.c_uint64)]


class CapsuleRow:
    """One named buffer of the live set: a uint8 numpy array + its valid-range rule."""

    def __init__(self, name, buf, fixed_bytes=0, bytes_per_token=0, n_seg=1, seg_stride=0):
        assert buf.dtype == np.uint8 and buf.flags["C_CONTIGUOUS"]
        self.name, self.buf = name, buf
        self.fixed_bytes, self.bytes_per_token = int(fixed_bytes), int(bytes_per_token)
        self.n_seg, self.seg_stride = int(n_seg), int(seg_stride)


def _table(rows):
    arr = (_Row * len(rows))()
    for i, r in enumerate(rows):
        arr[i] = _Row(r.buf.ctypes.data, r.buf.nbytes, r.fixed_bytes, r.bytes_per_token, r.n_seg, 0, r.seg_stride)
    return arr


def capsule_payload_bytes(rows, P):
    n = _load().esc_oracle_capsule_payload_bytes(_table(rows), len(rows), P)
    if n < 0:
        raise ValueError("capsule rows do not fit boundary P=%d" % P)
    return int(n)


def capsule_slab_bytes(rows, P):
    n = _load().esc_oracle_capsule_slab_bytes(_table(rows), len(rows), P)
    if n < 0:
        raise ValueError("capsule rows do not fit boundary P=%d" % P)
    return int(n)


def capsule_seg_offset(rows, P, row, seg):
    return int(_load().esc_oracle_capsule_seg_offset(_table(rows), len(rows), P, row, seg))


def capsule_snapshot(rows, P):
    """live rows -> new slab (uint8 array)."""
    slab = np.zeros(capsule_slab_bytes(rows, P), dtype=np.uint8)
    rc = _load().esc_oracle_capsule_snapshot(_table(rows), len(rows), P, slab.ctypes.data, slab.nbytes)
    if rc != 0:
        raise RuntimeError("capsule_snapshot rc=%d" % rc)
    return slab


def capsule_restore(rows, P, slab):
    """slab -> live rows, valid ranges only."""
    assert slab.dtype == np.uint8 and slab.flags["C_CONTIGUOUS"]
    rc = _load().esc_oracle_capsule_restore(_table(rows), len(rows), P, slab.ctypes.data, slab.nbytes)
    if rc != 0:
        raise RuntimeError("capsule_restore rc=%d" % rc)


def align_boundary(P, chunk):
    """P' = floor(P/C)*C."""
    return int(_load().esc_oracle_align_boundary(P, chunk))
