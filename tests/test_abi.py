"""CPU-only checks of the boundary: libesc.so builds for sm_100a, loads, exports every symbol
include/esc.h declares, and its pure host logic (no GPU compute) behaves as the header states."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def esc():
    from paper_2606_20537_b200 import build
    build.build()
    from paper_2606_20537_b200 import esc as m
    return m


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "esc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(esc_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_all_exported(esc):
    names = _declared_symbols()
    assert len(names) >= 24
    for n in names:
        assert hasattr(esc.lib, n), "libesc.so does not export %s" % n
    assert set(names) == set(esc.EXPORTS), "binding and header disagree: %s" % (set(names) ^ set(esc.EXPORTS))


def test_abi_version_and_strerror(esc):
    assert esc.abi_version() == 3        # 3: esc_scan_args.kind / .beta (delta-rule layers in a captured plan)
    for code in range(0, -7, -1):
        s = esc.strerror(code)
        assert s and "?" not in s
    assert "?" in esc.strerror(-99)


def test_align_boundary(esc):
    # P' = floor(P/C)*C
    assert esc.align_boundary(2048, 64) == 2048
    assert esc.align_boundary(2047, 64) == 1984
    assert esc.align_boundary(63, 64) == 0
    assert esc.align_boundary(16384 + 37, 128) == 16384
    assert esc.align_boundary(77, 0) == 77


def test_shape_key(esc):
    k1 = esc.shape_key_make(1, 16, 128, 128, esc.DTYPE_BF16, esc.DTYPE_F32, 64)
    k2 = esc.shape_key_make(1, 16, 128, 128, esc.DTYPE_BF16, esc.DTYPE_F32, 128)
    k3 = esc.shape_key_make(1, 16, 128, 128, esc.DTYPE_BF16, esc.DTYPE_BF16, 64)
    assert k1 and k2 and k3 and len({k1, k2, k3}) == 3
    assert esc.shape_key_make(1, 16, 128, 128, esc.DTYPE_BF16, esc.DTYPE_F32, 64) == k1   # deterministic, no T inside
    # unsupported combinations -> 0
    assert esc.shape_key_make(1, 16, 96, 128, esc.DTYPE_BF16, esc.DTYPE_F32, 64) == 0
    assert esc.shape_key_make(1, 16, 128, 128, esc.DTYPE_F32, esc.DTYPE_F32, 64) == 0
    assert esc.shape_key_make(1, 16, 128, 128, esc.DTYPE_BF16, esc.DTYPE_F32, 32) == 0
    assert esc.shape_key_make(0, 16, 128, 128, esc.DTYPE_BF16, esc.DTYPE_F32, 64) == 0


def test_null_handles_are_rejected(esc):
    assert esc.lib.esc_ctx_destroy(None) == esc.ERR_INVALID
    assert esc.lib.esc_bufset_destroy(None) == esc.ERR_INVALID
    assert esc.lib.esc_graph_destroy(None) == esc.ERR_INVALID
    assert esc.lib.esc_restore(None, None, None, None) == esc.ERR_INVALID
    assert esc.lib.esc_graph_launch(None, None) == esc.ERR_INVALID
    assert esc.lib.esc_linattn_scan(None, 0, *([None] * 7), 0, 0, 64, None) == esc.ERR_INVALID


def test_no_cpu_fallback(esc):
    """Without a CUDA device the product path must fail loudly (no CPU fallback)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(esc.EscError):
        esc.Ctx(0)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2606_20537_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "oracle/" not in txt and "_oracle.so" not in txt, f


def test_suffix_bucket_and_plan_key(esc):
    # the smallest chunk * 2^k >= T ("the suffix falls within a captured shape bucket")
    assert [esc.suffix_bucket(t, 64) for t in (0, 1, 64, 65, 128, 129, 1000, 4096)] == [0, 64, 64, 128, 128, 256, 1024, 4096]
    assert esc.suffix_bucket(100, 128) == 128 and esc.suffix_bucket(7, 0) == 7
    k = esc.shape_key_make(1, 16, 128, 128, esc.DTYPE_BF16, esc.DTYPE_F32, 64)
    keys = {esc.plan_key_make(k, b, P, n) for b in (64, 128) for P in (2048, 4096) for n in (1, 18)}
    assert len(keys) == 8 and esc.plan_key_make(k, 64, 2048, 18) in keys
    assert esc.lib.esc_plan_table_get(None, 1, None) == esc.ERR_INVALID
    assert esc.lib.esc_plan_table_set_capacity(None, 4) == esc.ERR_INVALID
