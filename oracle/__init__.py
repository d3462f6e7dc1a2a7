"""CPU oracle for the execution-state-capsule hot path.

ORACLE — TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
`cpu_baseline` / `--impl reference` legs may import this package.  The product package
(`paper_2606_20537_b200`) never imports it, and this package never imports the product.

What it holds (all pinned by `tests/test_oracle_*.py`, `-m "not gpu"`):
  * linattn_recurrence      fp64 sequential recurrence  S_t = g_t S_{t-1} + k_t^T v_t,
                            o_t = q_t S_t   (C, OpenMP across (b,h)) — north_star / SURVEY §8(c)
  * linattn_recurrence_np   the same definition restated in numpy (tiny shapes)
  * capsule_*               byte-level memcpy snapshot / restore of a named buffer set
                            (Algorithm 1)
  * fp8_stage.*             FP8 (E4M3) -> BF16 dequantisation stage (reading 23),
                            pinned by tests/test_oracle_fp8.py (format closed forms, torch float8_e4m3fn)
  * gdn_recurrence / causal_conv   gated delta rule and short causal convolution with carried window (the paper's
                            model family; reading 25), pinned by tests/test_oracle_gdn.py
Parity pins: closed form O(T^2), g==1 -> tril(QK^T)V (numpy matmul), scalar IIR
(scipy.signal.lfilter), hand example, linearity, restore-continue invariant; capsule ->
memcmp semantics and the size formula.  No function here is "parity unpinned".
"""
from . import fp8_stage  # noqa: F401
from .oracle import (  # noqa: F401
    bf16_bits_to_f32,
    linattn_recurrence,
    linattn_recurrence_np,
    gdn_recurrence,
    causal_conv,
    CapsuleRow,
    capsule_payload_bytes,
    capsule_slab_bytes,
    capsule_seg_offset,
    capsule_snapshot,
    capsule_restore,
    align_boundary,
    max_threads,
)
