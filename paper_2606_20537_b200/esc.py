"""ctypes binding of libesc.so — the C ABI declared in include/esc.h, same names.

Argument marshalling only: every step of the path (copy, scan, graph) runs in the library's
CUDA kernels.  torch is used by callers for device memory and streams; this module accepts
either torch tensors (their data_ptr()) or raw integer device addresses.  There is no CPU
fallback: if libesc.so is missing, importing this module raises.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("ESC_LIB") or os.path.join(_HERE, "libesc.so")   # ESC_LIB: another build of the same ABI

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "libesc.so is not built (%s). Run `python -m paper_2606_20537_b200.build` "
        "(nvcc, sm_100a). There is no CPU fallback." % LIB_PATH)

lib = C.CDLL(LIB_PATH)

OK, ERR_INVALID, ERR_UNALIGNED, ERR_MISMATCH, ERR_CAPACITY, ERR_UNSUPPORTED, ERR_CUDA = 0, -1, -2, -3, -4, -5, -6
DTYPE_BF16, DTYPE_F32 = 1, 2
SNAPSHOT_ALLOW_UNALIGNED = 1
MAX_FORK = 16
MAX_ROWS = 256
POSITION_UNKNOWN = 2**64 - 1
TIER_GPU, TIER_HOST = 0, 1
FORMAT_FP8_E4M3 = 1
ALL_ROWS = 2**32 - 1
RESTORE_DEQUANT_EAGER = 1
CONV_SILU = 1
SCAN_LINATTN, SCAN_GDN = 0, 1


class EscError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib.esc_strerror(code).decode()
        if code == ERR_CUDA:
            msg += " (cudaError %d)" % lib.esc_last_cuda_error()
        super().__init__("%s: %s" % (where, msg))


class BufDesc(C.Structure):
    _fields_ = [("name", C.c_char_p), ("dev_ptr", C.c_void_p), ("capacity_bytes", C.c_uint64),
                ("fixed_bytes", C.c_uint64), ("bytes_per_token", C.c_uint64), ("n_seg", C.c_uint32),
                ("reserved", C.c_uint32), ("seg_stride", C.c_uint64)]


class CapsuleInfo(C.Structure):
    _fields_ = [("boundary", C.c_uint64), ("chunk", C.c_uint64), ("slab_bytes", C.c_uint64),
                ("payload_bytes", C.c_uint64), ("layout_digest", C.c_uint64), ("prefix_digest", C.c_uint64),
                ("n_rows", C.c_uint32), ("n_segments", C.c_uint32), ("aligned", C.c_uint32), ("tier", C.c_uint32)]


class ScanArgs(C.Structure):
    _fields_ = [("key", C.c_uint64), ("q", C.c_void_p), ("k", C.c_void_p), ("v", C.c_void_p), ("g", C.c_void_p),
                ("state_in", C.c_void_p), ("state_out", C.c_void_p), ("o", C.c_void_p),
                ("T", C.c_uint64), ("t_stride", C.c_uint64), ("chunk", C.c_uint32), ("kind", C.c_uint32), ("beta", C.c_void_p)]


_P = C.c_void_p
_sig = {
    "esc_strerror": (C.c_char_p, [C.c_int]),
    "esc_abi_version": (C.c_uint32, []),
    "esc_last_cuda_error": (C.c_int, []),
    "esc_ctx_create": (C.c_int, [C.c_int, C.POINTER(_P)]),
    "esc_ctx_destroy": (C.c_int, [_P]),
    "esc_ctx_sm_count": (C.c_int, [_P, C.POINTER(C.c_int)]),
    "esc_bufset_create": (C.c_int, [_P, C.POINTER(BufDesc), C.c_uint32, C.POINTER(_P)]),
    "esc_bufset_destroy": (C.c_int, [_P]),
    "esc_bufset_layout_digest": (C.c_int, [_P, C.POINTER(C.c_uint64)]),
    "esc_bufset_set_position": (C.c_int, [_P, C.c_uint64]),
    "esc_bufset_get_position": (C.c_int, [_P, C.POINTER(C.c_uint64)]),
    "esc_capsule_bytes": (C.c_int, [_P, C.c_uint64, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]),
    "esc_align_boundary": (C.c_uint64, [C.c_uint64, C.c_uint64]),
    "esc_snapshot": (C.c_int, [_P, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint32, _P, C.c_uint64, _P, C.POINTER(_P)]),
    "esc_restore": (C.c_int, [_P, _P, C.POINTER(C.c_uint64), _P]),
    "esc_fork": (C.c_int, [_P, C.POINTER(_P), C.c_uint32, _P]),
    "esc_rollback": (C.c_int, [_P, _P, _P]),
    "esc_capsule_info_get": (C.c_int, [_P, C.POINTER(CapsuleInfo)]),
    "esc_capsule_demote": (C.c_int, [_P, _P, C.c_uint64, _P, C.POINTER(_P)]),
    "esc_capsule_promote": (C.c_int, [_P, _P, C.c_uint64, _P, C.POINTER(_P)]),
    "esc_bufset_attach_dequant_stage": (C.c_int, [_P, C.c_uint32, _P, C.c_uint64, C.c_uint32, C.c_float]),
    "esc_dequant_stage_valid_end": (C.c_int, [_P, C.c_uint32, C.POINTER(C.c_uint64)]),
    "esc_dequant_stage_fill": (C.c_int, [_P, C.c_uint32, C.c_uint64, _P]),
    "esc_restore_ex": (C.c_int, [_P, _P, C.POINTER(C.c_uint64), C.c_uint32, _P]),
    "esc_capsule_valid_end": (C.c_int, [_P, C.c_uint32, C.POINTER(C.c_uint64)]),
    "esc_restore_static_max_segments": (C.c_uint32, []),
    "esc_restore_static": (C.c_int, [_P, _P, C.POINTER(C.c_uint64), _P]),
    "esc_shape_key_make": (C.c_uint64, [C.c_uint32] * 7),
    "esc_scan_tile_columns": (C.c_int, [_P, C.c_uint64, C.POINTER(C.c_uint32)]),
    "esc_linattn_scan": (C.c_int, [_P, C.c_uint64] + [_P] * 7 + [C.c_uint64, C.c_uint64, C.c_uint32, _P]),
    "esc_gdn_scan": (C.c_int, [_P, C.c_uint64] + [_P] * 8 + [C.c_uint64, C.c_uint64, _P]),
    "esc_causal_conv": (C.c_int, [_P] * 6 + [C.c_uint32, C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _P]),
    "esc_graph_scratch_bytes": (C.c_uint64, []),
    "esc_graph_capture": (C.c_int, [_P, _P, C.c_uint64, C.POINTER(ScanArgs), C.c_uint32, _P, C.c_uint64, _P, C.POINTER(_P)]),
    "esc_graph_set_capsule": (C.c_int, [_P, _P, _P]),
    "esc_graph_launch": (C.c_int, [_P, _P]),
    "esc_graph_destroy": (C.c_int, [_P]),
    "esc_suffix_bucket": (C.c_uint64, [C.c_uint64, C.c_uint64]),
    "esc_plan_key_make": (C.c_uint64, [C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint32]),
    "esc_plan_table_set_capacity": (C.c_int, [_P, C.c_uint32]),
    "esc_plan_table_put": (C.c_int, [_P, C.c_uint64, _P]),
    "esc_plan_table_get": (C.c_int, [_P, C.c_uint64, C.POINTER(_P)]),
    "esc_plan_table_contains": (C.c_int, [_P, C.c_uint64, C.POINTER(C.c_uint32)]),
    "esc_plan_table_stats": (C.c_int, [_P, C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_uint64),
                                       C.POINTER(C.c_uint64)]),
}
for _n, (_r, _a) in _sig.items():
    _f = getattr(lib, _n)
    _f.restype, _f.argtypes = _r, _a
EXPORTS = tuple(_sig)


def _check(rc, where):
    if rc != OK:
        raise EscError(rc, where)


def _ptr(x):
    """torch tensor / int / None -> device address (int or None)."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    return x.data_ptr()


def _stream(s):
    """torch.cuda.Stream / int / None -> cudaStream_t value."""
    if s is None:
        return None
    if isinstance(s, int):
        return s or None
    return s.cuda_stream or None


def strerror(code):
    return lib.esc_strerror(code).decode()


def abi_version():
    return int(lib.esc_abi_version())


def align_boundary(P, chunk):
    return int(lib.esc_align_boundary(P, chunk))


def shape_key_make(B, H, d_k, d_v, in_dtype=DTYPE_BF16, out_dtype=DTYPE_F32, chunk=64):
    return int(lib.esc_shape_key_make(B, H, d_k, d_v, in_dtype, out_dtype, chunk))


class Ctx:
    def __init__(self, device=0):
        h = _P()
        _check(lib.esc_ctx_create(device, C.byref(h)), "esc_ctx_create")
        self.h = h

    @property
    def sm_count(self):
        n = C.c_int()
        _check(lib.esc_ctx_sm_count(self.h, C.byref(n)), "esc_ctx_sm_count")
        return n.value

    # Graph[key] table (bounded, LRU): the context owns the plans put into it
    def _reconcile_plans(self):
        """Drop the python wrappers of plans the C table no longer holds (LRU eviction, capacity shrink, replacement):
        their handles are dead, and their buffers need not be kept alive any longer."""
        plans = getattr(self, "_plans", {})
        for key in list(plans):
            present = C.c_uint32()
            _check(lib.esc_plan_table_contains(self.h, key, C.byref(present)), "esc_plan_table_contains")
            if not present.value:
                g = plans.pop(key)
                g.h = None          # launch() / set_capsule() on an evicted plan now fail in python instead of in C
                g._keep = ()

    def plan_table_set_capacity(self, n):
        _check(lib.esc_plan_table_set_capacity(self.h, n), "esc_plan_table_set_capacity")
        self._reconcile_plans()

    def plan_put(self, plan_key, graph):
        _check(lib.esc_plan_table_put(self.h, plan_key, graph.h), "esc_plan_table_put")
        graph.owned = False
        self._plans = getattr(self, "_plans", {})
        old = self._plans.get(plan_key)
        if old is not None and old is not graph:
            old.h, old._keep = None, ()
        self._plans[plan_key] = graph   # keeps the python references (buffers) of the plan alive
        self._reconcile_plans()

    def plan_get(self, plan_key):
        """The captured plan or None ("a new shape needing capture")."""
        h = _P()
        rc = lib.esc_plan_table_get(self.h, plan_key, C.byref(h))
        if rc == ERR_MISMATCH:
            return None
        _check(rc, "esc_plan_table_get")
        g = getattr(self, "_plans", {}).get(plan_key)
        return g if g is not None and g.h and g.h.value == h.value else Graph(h, owned=False)

    def plan_stats(self):
        n, a, b, c = C.c_uint32(), C.c_uint64(), C.c_uint64(), C.c_uint64()
        _check(lib.esc_plan_table_stats(self.h, C.byref(n), C.byref(a), C.byref(b), C.byref(c)), "esc_plan_table_stats")
        return {"size": n.value, "hits": a.value, "misses": b.value, "evictions": c.value}

    def close(self):
        if self.h:
            for g in getattr(self, "_plans", {}).values():
                g.h, g._keep = None, ()
            self._plans = {}
            lib.esc_ctx_destroy(self.h)
            self.h = None


class BufSet:
    """A live set (esc_bufset_create) or a capsule (returned by snapshot)."""

    def __init__(self, handle, keep=()):
        self.h = handle
        self._keep = keep   # python references that must outlive the handle (tensors, slab)

    @property
    def layout_digest(self):
        d = C.c_uint64()
        _check(lib.esc_bufset_layout_digest(self.h, C.byref(d)), "esc_bufset_layout_digest")
        return d.value

    @property
    def position(self):
        p = C.c_uint64()
        _check(lib.esc_bufset_get_position(self.h, C.byref(p)), "esc_bufset_get_position")
        return p.value

    def set_position(self, P):
        _check(lib.esc_bufset_set_position(self.h, P), "esc_bufset_set_position")

    def capsule_bytes(self, P):
        a, b = C.c_uint64(), C.c_uint64()
        _check(lib.esc_capsule_bytes(self.h, P, C.byref(a), C.byref(b)), "esc_capsule_bytes")
        return a.value, b.value

    def info(self):
        i = CapsuleInfo()
        _check(lib.esc_capsule_info_get(self.h, C.byref(i)), "esc_capsule_info_get")
        return i

    def valid_end(self, row):
        n = C.c_uint64()
        _check(lib.esc_capsule_valid_end(self.h, row, C.byref(n)), "esc_capsule_valid_end")
        return n.value

    def attach_dequant_stage(self, row, stage, scale=1.0, fmt=FORMAT_FP8_E4M3, stage_bytes=None):
        """stage: torch bf16/uint8 tensor (or device address + stage_bytes) shaped like the FP8 row, 2 bytes per code."""
        if stage_bytes is None:
            stage_bytes = stage.numel() * stage.element_size()
        _check(lib.esc_bufset_attach_dequant_stage(self.h, row, _ptr(stage), stage_bytes, fmt, scale),
               "esc_bufset_attach_dequant_stage")
        self._keep = tuple(self._keep) + (stage,)

    def stage_valid_end(self, row):
        n = C.c_uint64()
        _check(lib.esc_dequant_stage_valid_end(self.h, row, C.byref(n)), "esc_dequant_stage_valid_end")
        return n.value

    def stage_fill(self, row, upto_tokens, stream=None):
        _check(lib.esc_dequant_stage_fill(self.h, row, upto_tokens, _stream(stream)), "esc_dequant_stage_fill")

    def destroy(self):
        if self.h:
            lib.esc_bufset_destroy(self.h)
            self.h = None
            self._keep = ()


def bufset_create(ctx, rows):
    """rows: iterable of (name, tensor_or_addr, capacity_bytes, fixed_bytes, bytes_per_token, n_seg, seg_stride)."""
    rows = list(rows)
    arr = (BufDesc * len(rows))()
    for i, (name, buf, cap, fixed, per_tok, n_seg, stride) in enumerate(rows):
        arr[i] = BufDesc(name.encode(), _ptr(buf), cap, fixed, per_tok, n_seg, 0, stride)
    h = _P()
    _check(lib.esc_bufset_create(ctx.h, arr, len(rows), C.byref(h)), "esc_bufset_create")
    return BufSet(h, keep=tuple(r[1] for r in rows))


def snapshot(live, P, chunk, storage, storage_bytes=None, prefix_digest=0, flags=0, stream=None):
    """storage: torch uint8 tensor (or address + storage_bytes). Returns the capsule BufSet."""
    if storage_bytes is None:
        storage_bytes = storage.numel() * storage.element_size()
    h = _P()
    _check(lib.esc_snapshot(live.h, P, chunk, prefix_digest, flags, _ptr(storage), storage_bytes, _stream(stream),
                            C.byref(h)), "esc_snapshot")
    return BufSet(h, keep=(storage,))


def restore(live, capsule, expect_prefix_digest=None, stream=None):
    e = None if expect_prefix_digest is None else C.byref(C.c_uint64(expect_prefix_digest))
    _check(lib.esc_restore(live.h, capsule.h, e, _stream(stream)), "esc_restore")


def restore_static(live, capsule, expect_prefix_digest=None, stream=None):
    """esc_restore with its descriptor tables in the library's static device array: no scratch, no device allocation."""
    e = None if expect_prefix_digest is None else C.byref(C.c_uint64(expect_prefix_digest))
    _check(lib.esc_restore_static(live.h, capsule.h, e, _stream(stream)), "esc_restore_static")


def restore_ex(live, capsule, expect_prefix_digest=None, flags=0, stream=None):
    e = None if expect_prefix_digest is None else C.byref(C.c_uint64(expect_prefix_digest))
    _check(lib.esc_restore_ex(live.h, capsule.h, e, flags, _stream(stream)), "esc_restore_ex")


def fork(capsule, lives, stream=None):
    arr = (_P * len(lives))(*[l.h for l in lives])
    _check(lib.esc_fork(capsule.h, arr, len(lives), _stream(stream)), "esc_fork")


def capsule_demote(capsule, storage_host, storage_bytes=None, stream=None):
    """storage_host: pinned torch uint8 tensor (or host address + storage_bytes). Returns the HOST-tier capsule."""
    if storage_bytes is None:
        storage_bytes = storage_host.numel() * storage_host.element_size()
    h = _P()
    _check(lib.esc_capsule_demote(capsule.h, _ptr(storage_host), storage_bytes, _stream(stream), C.byref(h)),
           "esc_capsule_demote")
    return BufSet(h, keep=(storage_host,))


def capsule_promote(host_capsule, storage_dev, storage_bytes=None, stream=None):
    if storage_bytes is None:
        storage_bytes = storage_dev.numel() * storage_dev.element_size()
    h = _P()
    _check(lib.esc_capsule_promote(host_capsule.h, _ptr(storage_dev), storage_bytes, _stream(stream), C.byref(h)),
           "esc_capsule_promote")
    return BufSet(h, keep=(storage_dev,))


def rollback(live, capsule_earlier, stream=None):
    _check(lib.esc_rollback(live.h, capsule_earlier.h, _stream(stream)), "esc_rollback")


def scan_tile_columns(ctx, key):
    w = C.c_uint32()
    _check(lib.esc_scan_tile_columns(ctx.h, key, C.byref(w)), "esc_scan_tile_columns")
    return w.value


def linattn_scan(ctx, key, q, k, v, g, state_in, state_out, o, T, t_stride, chunk, stream=None):
    _check(lib.esc_linattn_scan(ctx.h, key, _ptr(q), _ptr(k), _ptr(v), _ptr(g), _ptr(state_in), _ptr(state_out),
                                _ptr(o), T, t_stride, chunk, _stream(stream)), "esc_linattn_scan")


def gdn_scan(ctx, key, q, k, v, g, beta, state_in, state_out, o, T, t_stride, stream=None):
    _check(lib.esc_gdn_scan(ctx.h, key, _ptr(q), _ptr(k), _ptr(v), _ptr(g), _ptr(beta), _ptr(state_in), _ptr(state_out),
                            _ptr(o), T, t_stride, _stream(stream)), "esc_gdn_scan")


def causal_conv(ctx, x, w, state_in, state_out, y, B, T, t_stride, Cch, W, flags=0, stream=None):
    _check(lib.esc_causal_conv(ctx.h, _ptr(x), _ptr(w), _ptr(state_in), _ptr(state_out), _ptr(y), B, T, t_stride, Cch, W,
                               flags, _stream(stream)), "esc_causal_conv")


def scan_args(key, q, k, v, g, state_in, state_out, o, T, t_stride, chunk, beta=None):
    """One layer of a captured plan: a linear-attention scan, or (beta given) a gated delta-rule scan."""
    a = ScanArgs(key, _ptr(q), _ptr(k), _ptr(v), _ptr(g), _ptr(state_in), _ptr(state_out), _ptr(o),
                 T, t_stride, chunk, SCAN_LINATTN if beta is None else SCAN_GDN, _ptr(beta))
    a._keep = (q, k, v, g, state_in, state_out, o, beta)   # the struct holds raw addresses: keep the tensors alive with it
    return a


def suffix_bucket(T, chunk):
    return int(lib.esc_suffix_bucket(T, chunk))


def plan_key_make(shape_key, bucket, max_boundary, n_layers):
    return int(lib.esc_plan_key_make(shape_key, bucket, max_boundary, n_layers))


class Graph:
    def __init__(self, handle, keep=(), owned=True):
        self.h = handle
        self._keep = keep
        self.owned = owned      # False once a context's plan table owns the handle

    def _handle(self, where):
        if not self.h:
            raise EscError(ERR_INVALID, where + " (plan destroyed or evicted from the Graph[key] table)")
        return self.h

    def set_capsule(self, capsule, stream=None):
        _check(lib.esc_graph_set_capsule(self._handle("esc_graph_set_capsule"), capsule.h, _stream(stream)),
               "esc_graph_set_capsule")

    def launch(self, stream=None):
        _check(lib.esc_graph_launch(self._handle("esc_graph_launch"), _stream(stream)), "esc_graph_launch")

    def destroy(self):
        if self.h and self.owned:
            lib.esc_graph_destroy(self.h)
        if self.owned:
            self.h = None
            self._keep = ()


def graph_scratch_bytes():
    return int(lib.esc_graph_scratch_bytes())


def graph_capture(ctx, live, max_boundary, layers, stream, scratch=None):
    """layers: list of ScanArgs; live may be None (cold plan).  stream must be a non-default stream.
    scratch: caller-owned device memory (torch uint8 tensor) of graph_scratch_bytes() for the restore node's descriptor
    table; allocated here with torch when omitted (the library itself never allocates device memory)."""
    arr = (ScanArgs * max(1, len(layers)))(*layers)
    h = _P()
    nbytes = 0
    if live is not None:
        if scratch is None:
            import torch
            dev = stream.device if hasattr(stream, "device") else "cuda"
            scratch = torch.empty(graph_scratch_bytes(), dtype=torch.uint8, device=dev)
        nbytes = scratch.numel() * scratch.element_size() if hasattr(scratch, "numel") else graph_scratch_bytes()
    _check(lib.esc_graph_capture(ctx.h, live.h if live is not None else None, max_boundary, arr, len(layers),
                                 _ptr(scratch) if live is not None else None, nbytes, _stream(stream), C.byref(h)),
           "esc_graph_capture")
    return Graph(h, keep=(live, tuple(layers), scratch))
