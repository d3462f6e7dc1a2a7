"""Shared plumbing of the -m gpu parity tests: torch allocations for a synth layout, host twins
for the oracle, integer-view comparisons, the tolerance metrics of DESIGN.md.  Holds none of
the method's arithmetic."""
import numpy as np
import torch

import oracle
from paper_2606_20537_b200 import synth

DEV = "cuda:0"

# north_star tolerances under the metric readings of DESIGN.md (#7, #8)
TOL_O = 2e-3      # ||o_gpu - o_ref||_inf / ||o_ref||_inf
TOL_S = 1e-3      # ||S_gpu - S_ref||_F / ||S_ref||_F


def esc_mod():
    from paper_2606_20537_b200 import esc   # raises loudly when libesc.so is missing
    return esc


def to_dev(a: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def dev_bytes(t: torch.Tensor) -> np.ndarray:
    """device tensor -> host uint8 view of its bytes (integer compare: NaN-safe, -0 != +0)."""
    return t.contiguous().view(torch.uint8).cpu().numpy()


class LiveSet:
    """One live buffer set on the GPU (torch uint8 tensors) + the same bytes on the host."""

    def __init__(self, esc, ctx, specs, seed_ids, offset_bytes=0):
        self.specs = specs
        self.host = [synth.random_bytes(s.capacity_bytes, *seed_ids, i) for i, s in enumerate(specs)]
        self.base = [torch.empty(s.capacity_bytes + offset_bytes, dtype=torch.uint8, device=DEV) for s in specs]
        self.dev = [b[offset_bytes:] for b in self.base]
        for d, h in zip(self.dev, self.host):
            d.copy_(torch.from_numpy(h))
        self.set = esc.bufset_create(ctx, [(s.name, d, s.capacity_bytes, s.fixed_bytes, s.bytes_per_token, s.n_seg,
                                            s.seg_stride) for s, d in zip(specs, self.dev)])

    def oracle_rows(self):
        return [oracle.CapsuleRow(s.name, h, s.fixed_bytes, s.bytes_per_token, s.n_seg, s.seg_stride)
                for s, h in zip(self.specs, self.host)]

    def fill(self, *seed_ids, pattern=None):
        """Overwrite every live buffer (device and host twin) — the 'dirty' step."""
        for i, (d, s) in enumerate(zip(self.dev, self.specs)):
            if pattern is None:
                self.host[i] = synth.random_bytes(s.capacity_bytes, *seed_ids, i)
            else:
                self.host[i] = np.full(s.capacity_bytes, pattern, np.uint8)
            d.copy_(torch.from_numpy(self.host[i]))

    def set_row(self, i, arr: np.ndarray):
        """Overwrite the head of row i (device + host twin) with the bytes of `arr`."""
        b = np.ascontiguousarray(arr).view(np.uint8).reshape(-1)
        self.host[i][: b.size] = b
        self.dev[i][: b.size].copy_(torch.from_numpy(b))

    def assert_equals_host(self):
        torch.cuda.synchronize()
        for d, h, s in zip(self.dev, self.host, self.specs):
            got = d.cpu().numpy()
            assert np.array_equal(got, h), "row %s differs from the oracle's bytes" % s.name


def scan_dev_inputs(si: synth.ScanInputs):
    q = to_dev(si.q_bits.view(np.int16)).view(torch.bfloat16)
    k = to_dev(si.k_bits.view(np.int16)).view(torch.bfloat16)
    v = to_dev(si.v_bits.view(np.int16)).view(torch.bfloat16)
    g = to_dev(si.g)
    return q, k, v, g


def err_o(o_gpu, o_ref):
    o_gpu = np.asarray(o_gpu, np.float64)
    den = np.abs(o_ref).max()
    return float(np.abs(o_gpu - o_ref).max() / den) if den > 0 else float(np.abs(o_gpu).max())


def err_s(s_gpu, s_ref):
    s_gpu = np.asarray(s_gpu, np.float64)
    den = np.linalg.norm(s_ref.ravel())
    return float(np.linalg.norm((s_gpu - s_ref).ravel()) / den) if den > 0 else float(np.abs(s_gpu).max())


TOL_S_SLICE = 2e-3   # the same ratio over each (b, h, 16-column d_v slice) — the kernels' unit of work


def err_s_slices(s_gpu, s_ref, width=16):
    """max over (b, h, d_v slice of `width` columns) of the relative Frobenius error of that slice: a defect confined
    to one CTA's slice of one head is not diluted by the rest of the layer."""
    s_gpu = np.asarray(s_gpu, np.float64)
    s_ref = np.asarray(s_ref, np.float64)
    B, H, dk, dv = s_ref.shape
    w = min(width, dv)
    d = (s_gpu - s_ref).reshape(B, H, dk, dv // w, w)
    r = s_ref.reshape(B, H, dk, dv // w, w)
    num = np.sqrt((d * d).sum(axis=(2, 4)))
    den = np.sqrt((r * r).sum(axis=(2, 4)))
    tiny = den <= 0
    return float(np.where(tiny, num, num / np.where(tiny, 1.0, den)).max())


def assert_state_close(s_gpu, s_ref, tag=""):
    """north_star's state gate (whole-layer relative Frobenius <= 1e-3) plus the per-slice maximum (<= 2e-3)."""
    s_gpu = s_gpu.cpu().numpy() if hasattr(s_gpu, "cpu") else s_gpu
    e = err_s(s_gpu, s_ref)
    assert e <= TOL_S, "S error %.3e %s" % (e, tag)
    es = err_s_slices(s_gpu, s_ref)
    assert es <= TOL_S_SLICE, "S per-slice error %.3e %s" % (es, tag)


def sample_heads(B, H, n, *seed_ids):
    """n distinct seeded (b, h) pairs (the full-size tests check a sample of heads against the oracle)."""
    r = synth.rng(900, *seed_ids)
    idx = r.choice(B * H, size=min(n, B * H), replace=False)
    return [(int(i) // H, int(i) % H) for i in idx]


def bits_equal(a: torch.Tensor, b: torch.Tensor) -> bool:
    return bool(torch.equal(a.contiguous().view(torch.uint8), b.contiguous().view(torch.uint8)))
