"""Pins for the capsule oracle (CPU only): the memcpy definition (byte equality via plain numpy
slicing written out here, not via the oracle), the paper's printed size table, alignment rule."""
import os

import numpy as np
import pytest

import oracle
from paper_2606_20537_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_table7_capsule_sizes.txt")


def _mk_rows(specs, seed):
    rows = []
    for i, s in enumerate(specs):
        buf = synth.random_bytes(s.capacity_bytes, 901, seed, i)
        rows.append(oracle.CapsuleRow(s.name, buf, s.fixed_bytes, s.bytes_per_token, s.n_seg, s.seg_stride))
    return rows


def _valid_ranges(r, P):
    n = r.fixed_bytes + P * r.bytes_per_token
    return [(s * r.seg_stride, s * r.seg_stride + n) for s in range(r.n_seg)]


SMALL = [
    synth.RowSpec("state", 4096, fixed_bytes=4096),
    synth.RowSpec("robot640", 640, fixed_bytes=640),                                   # one 640-byte buffer
    synth.RowSpec("odd", 1000, fixed_bytes=997),                                       # byte-granular tail
    synth.RowSpec("kv_tok", 64 * 24, bytes_per_token=24),                               # token-major
    synth.RowSpec("kv_head", 4 * 64 * 10, bytes_per_token=10, n_seg=4, seg_stride=640), # head-major, odd seg bytes
    synth.RowSpec("mixed", 300 + 64 * 3, fixed_bytes=300, bytes_per_token=3),
]


def test_paper_table7_sizes_golden():
    # PAPER.md:249-252 Table 7: 160/224/352/608 MiB at 2k/4k/8k/16k = 96 MiB fixed + 32 KiB/token.
    pts = [tuple(int(x) for x in ln.split()) for ln in open(GOLDEN) if ln.strip() and not ln.startswith("#")]
    assert len(pts) == 4
    fixed, per_tok = 96 << 20, 32 << 10
    from oracle import oracle as impl
    stand_in = np.zeros(1, np.uint8)   # the size query touches no bytes; capacities are set on the table below
    tab = impl._table([oracle.CapsuleRow("fixed", stand_in, fixed_bytes=fixed),
                       oracle.CapsuleRow("kv", stand_in, bytes_per_token=per_tok)])
    tab[0].capacity_bytes = fixed
    tab[1].capacity_bytes = per_tok * 16384
    for P, mib in pts:
        assert impl._load().esc_oracle_capsule_payload_bytes(tab, 2, P) == mib << 20


def test_hybrid_layout_sizes_match_survey_table():
    # SURVEY.md §8 geometry table: 18 MiB fold states + 24 KiB/token of bf16 KV
    expect = {2048: 69206016, 4096: 119537664, 8192: 220200960, 16384: 421527552}
    specs = synth.hybrid_layout(16384)
    assert len(specs) == 18 + 12
    fixed = sum(s.fixed_bytes for s in specs)
    per_tok = sum(s.bytes_per_token * s.n_seg for s in specs)
    assert fixed == 18 << 20 and per_tok == 24 << 10
    for P, nbytes in expect.items():
        assert fixed + P * per_tok == nbytes
    for hm in (False, True):
        for packed in (False, True):
            sp = synth.hybrid_layout(4096, head_major=hm, packed_kv=packed)
            assert sum(s.bytes_per_token * s.n_seg for s in sp) == 24 << 10


@pytest.mark.parametrize("P", [0, 1, 17, 64])
def test_snapshot_restore_is_memcpy_of_valid_ranges(P):
    rows = _mk_rows(SMALL, seed=P)
    orig = [r.buf.copy() for r in rows]
    payload = oracle.capsule_payload_bytes(rows, P)
    assert payload == sum(r.n_seg * (r.fixed_bytes + P * r.bytes_per_token) for r in rows)
    slab = oracle.capsule_snapshot(rows, P)
    assert slab.nbytes == oracle.capsule_slab_bytes(rows, P) >= payload
    # slab holds each valid range at a 16-B aligned offset, rows 256-B aligned, in table order
    last = -1
    for i, r in enumerate(rows):
        for s, (a, b) in enumerate(_valid_ranges(r, P)):
            off = oracle.capsule_seg_offset(rows, P, i, s)
            assert off % 16 == 0 and off > last - 1 and (s > 0 or off % 256 == 0)
            assert np.array_equal(slab[off:off + (b - a)], orig[i][a:b])
            last = off + (b - a)
    # dirty every live byte, restore: valid ranges equal the originals, the rest keeps the dirt (reading #14)
    for r in rows:
        r.buf[:] = 0xA5
    oracle.capsule_restore(rows, P, slab)
    for i, r in enumerate(rows):
        mask = np.zeros(r.buf.nbytes, bool)
        for a, b in _valid_ranges(r, P):
            mask[a:b] = True
        assert np.array_equal(r.buf[mask], orig[i][mask])
        assert np.all(r.buf[~mask] == 0xA5)


def test_capacity_overflow_is_rejected():
    rows = _mk_rows(SMALL, seed=1)
    with pytest.raises(ValueError):
        oracle.capsule_slab_bytes(rows, 65)   # kv_tok holds 64 tokens


def test_align_boundary():
    # PAPER.md:118  P' = floor(P/C)*C
    assert [oracle.align_boundary(P, 64) for P in (0, 1, 63, 64, 65, 2047, 2048, 16384 + 37)] == [0, 0, 0, 64, 64, 1984, 2048, 16384]
    assert oracle.align_boundary(185, 128) == 128
