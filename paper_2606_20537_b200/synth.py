"""Seeded synthetic inputs shaped like the paper's hybrid-model workloads.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.  It holds
none of the method's arithmetic (no recurrence, no chunk algebra, no copy logic): only
random draws, the input-side rounding to bf16, and the buffer-set geometry of the configs
in BASELINE.json.  Recipe: SURVEY.md §8(d) "Concrete synthetic inputs", DESIGN.md "Inputs".

The paper's own workload (Table 7: a hybrid linear-/full-attention LLM,
prefixes 2k-16k, short suffix) is not available; these inputs take its *shape* and stand in.
"""
from dataclasses import dataclass

import numpy as np

BASE_SEED = 20537


def rng(*ids) -> np.random.Generator:
    """numpy Generator seeded by (BASE_SEED, *ids) — e.g. rng(config, layer, session, tensor_id)."""
    return np.random.default_rng([BASE_SEED, *[int(i) for i in ids]])


# ---------------------------------------------------------------------------------------
# input-side dtype plumbing (bit-level, exact)
# ---------------------------------------------------------------------------------------
def f32_to_bf16_bits(x) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns (finite inputs)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32).astype(np.uint64)
    r = (u + np.uint64(0x7FFF) + ((u >> np.uint64(16)) & np.uint64(1))) >> np.uint64(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(bits) -> np.ndarray:
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32)


# ---------------------------------------------------------------------------------------
# scan inputs
# ---------------------------------------------------------------------------------------
GATE_MEAN = {"fast": 0.0, "slow": -4.0}   # x ~ N(mean, 1); g = exp(-softplus(x)) = sigmoid(-x)


@dataclass
class ScanInputs:
    q_bits: np.ndarray   # uint16 [B,T,H,dk]  bf16 bit patterns
    k_bits: np.ndarray   # uint16 [B,T,H,dk]
    v_bits: np.ndarray   # uint16 [B,T,H,dv]
    g: np.ndarray        # float32 [B,T,H], in (0,1]

    @property
    def shape(self):
        B, T, H, dk = self.q_bits.shape
        return B, T, H, dk, self.v_bits.shape[-1]

    def as_f32(self):
        """fp32 containers holding the exact bf16 values (what the oracle consumes)."""
        return (bf16_bits_to_f32(self.q_bits), bf16_bits_to_f32(self.k_bits),
                bf16_bits_to_f32(self.v_bits), self.g)


def scan_inputs(B, T, H, dk, dv, seed_ids=(0,), gate="fast") -> ScanInputs:
    """q,k ~ N(0,1) L2-normalised per (b,t,h) over dk, v ~ N(0,1), all rounded once to bf16;
    g = exp(-softplus(x)), x ~ N(mean,1) per (b,t,h), computed in fp64 and rounded once to fp32.
    gate: "fast" (x~N(0,1), the BASELINE.json distribution), "slow" (x~N(-4,1), g~0.97),
    "one" (g == 1)."""
    r = rng(*seed_ids)
    q = r.standard_normal((B, T, H, dk))
    k = r.standard_normal((B, T, H, dk))
    v = r.standard_normal((B, T, H, dv))
    q /= np.linalg.norm(q, axis=-1, keepdims=True)
    k /= np.linalg.norm(k, axis=-1, keepdims=True)
    if gate == "one":
        g = np.ones((B, T, H), dtype=np.float32)
        r.standard_normal((B, T, H))  # keep the stream position independent of the gate kind
    else:
        x = r.standard_normal((B, T, H)) + GATE_MEAN[gate]
        g = np.exp(-np.logaddexp(0.0, x)).astype(np.float32)
        g = np.maximum(g, np.float32(1e-30))  # contract: g in (0,1]
    return ScanInputs(f32_to_bf16_bits(q), f32_to_bf16_bits(k), f32_to_bf16_bits(v), g)


def gdn_beta(B, T, H, seed_ids=(0,)) -> np.ndarray:
    """Write strengths of the gated delta rule (reading 25): beta = sigmoid(x), x ~ N(0,1) per (b,t,h), fp32."""
    x = rng(*seed_ids, 555).standard_normal((B, T, H))
    return (1.0 / (1.0 + np.exp(-x))).astype(np.float32)


def conv_inputs(B, T, C, W, seed_ids=(0,)):
    """Short causal convolution inputs: x ~ N(0,1) rounded once to bf16 (bits, uint16 [B,T,C]); taps w ~ N(0,1)/sqrt(W)
    fp32 [C,W]; a carried window of W-1 earlier bf16-representable inputs as fp32 [B,C,W-1]."""
    r = rng(*seed_ids, 556)
    x_bits = f32_to_bf16_bits(r.standard_normal((B, T, C)))
    w = (r.standard_normal((C, W)) / np.sqrt(W)).astype(np.float32)
    st = bf16_bits_to_f32(f32_to_bf16_bits(r.standard_normal((B, C, max(W - 1, 0))))).astype(np.float32)
    return x_bits, w, st


def scan_state(B, H, dk, dv, seed_ids=(0,), scale=1.0) -> np.ndarray:
    """A non-zero fp32 start state [B,H,dk,dv] (for S_0 != 0 cases)."""
    return (rng(*seed_ids, 777).standard_normal((B, H, dk, dv)) * scale).astype(np.float32)


# ---------------------------------------------------------------------------------------
# capsule buffer-set geometry
# ---------------------------------------------------------------------------------------
@dataclass
class RowSpec:
    name: str
    capacity_bytes: int
    fixed_bytes: int = 0
    bytes_per_token: int = 0
    n_seg: int = 1
    seg_stride: int = 0


def hybrid_layout(t_max, n_linear=18, n_full=6, H=16, dk=128, dv=128, kv_heads=4, head_dim=256,
                  kv_elem_bytes=2, head_major=False, packed_kv=False):
    """The 24-layer hybrid buffer set of BASELINE.json configs 1-3 (SURVEY.md §8 geometry):
    n_linear fold states fp32 [H,dk,dv] (fixed) + n_full full-attention layers' contiguous
    K and V buffers (bf16, token-major [t_max, kv_heads, head_dim], or head-major
    [kv_heads, t_max, head_dim] -> n_seg = kv_heads)."""
    rows = []
    per_tok = kv_heads * head_dim * kv_elem_bytes
    li = fi = 0
    # interleave like a hybrid stack: every 4th layer is full attention (3 linear : 1 full)
    period = (n_linear + n_full) // n_full if n_full else 0
    for layer in range(n_linear + n_full):
        is_full = n_full and (layer % period == period - 1) and fi < n_full
        if is_full:
            names = ["kv"] if packed_kv else ["k", "v"]
            for nm in names:
                mult = 2 if packed_kv else 1
                if head_major:
                    seg = t_max * head_dim * kv_elem_bytes * mult
                    rows.append(RowSpec(f"L{layer:02d}.full.{nm}", seg * kv_heads, 0,
                                        head_dim * kv_elem_bytes * mult, kv_heads, seg))
                else:
                    rows.append(RowSpec(f"L{layer:02d}.full.{nm}", t_max * per_tok * mult, 0, per_tok * mult, 1, 0))
            fi += 1
        else:
            rows.append(RowSpec(f"L{layer:02d}.lin.state", H * dk * dv * 4, H * dk * dv * 4, 0, 1, 0))
            li += 1
    return rows


def random_bytes(n, *seed_ids) -> np.ndarray:
    """n seeded random bytes (uint8)."""
    r = rng(*seed_ids)
    out = np.empty(n, dtype=np.uint8)
    nw = n // 8
    if nw:
        out[: nw * 8].view(np.uint64)[:] = r.integers(0, 2**64, size=nw, dtype=np.uint64)
    if n - nw * 8:
        out[nw * 8:] = r.integers(0, 256, size=n - nw * 8, dtype=np.uint8)
    return out
