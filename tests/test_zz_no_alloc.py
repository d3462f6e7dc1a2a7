"""-m gpu: esc_restore_static — restore with its descriptor tables in the library's static device array (no caller scratch,
no device allocation; include/esc.h) — against the existing esc_restore path and the byte-level memcpy oracle.  Bar: bit-exact.

Collected last on purpose (the suite runs with pytest -x: a failure here hides nothing after it).  Every test makes two calls in
a row on the shared static tables, so it passes alone in a fresh process and after the other tests have used the library."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_20537_b200 import synth
from gpu_util import DEV, LiveSet, esc_mod

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def esc():
    return esc_mod()


@pytest.fixture(scope="module")
def ctx(esc):
    c = esc.Ctx(0)
    yield c
    c.close()


def _snapshot(esc, live, P, chunk=0):
    slab = torch.zeros(live.set.capsule_bytes(P)[0], dtype=torch.uint8, device=DEV)   # (padding between segments is never written)
    cap = esc.snapshot(live.set, P, chunk, slab, prefix_digest=0x5EED + P)
    torch.cuda.synchronize()
    return cap, slab


def _two_restores_match(esc, ctx, specs, P1, P2, seed):
    """Two identical live sets: A goes through esc_restore (the existing path), B through esc_restore_static, twice in a row with
    capsules of different boundaries (the second call finds the first call's tables in the static array)."""
    a = LiveSet(esc, ctx, specs, (seed,))
    b = LiveSet(esc, ctx, specs, (seed,))
    caps = []
    for P in (P1, P2):
        a.fill(seed, P)
        b.fill(seed, P)
        cap_a, slab_a = _snapshot(esc, a, P)
        cap_b, slab_b = _snapshot(esc, b, P)
        assert torch.equal(slab_a, slab_b)
        caps.append((P, cap_a, slab_a, cap_b, slab_b))
    for rnd, (P, cap_a, slab_a, cap_b, slab_b) in enumerate(caps):
        ref_slab = slab_a.cpu().numpy()
        for pat in (None, 0xFF):   # adversarial dirty: another run's bytes, then NaN patterns
            a.fill(900 + rnd, P, pattern=pat)
            b.fill(900 + rnd, P, pattern=pat)
            esc.restore(a.set, cap_a, expect_prefix_digest=0x5EED + P)
            esc.restore_static(b.set, cap_b, expect_prefix_digest=0x5EED + P)
            torch.cuda.synchronize()
            for da, db, s in zip(a.dev, b.dev, specs):
                assert torch.equal(da, db), "row %s: static-table restore differs from esc_restore" % s.name
            oracle.capsule_restore(b.oracle_rows(), P, ref_slab)   # and both equal the oracle's memcpy restore
            b.assert_equals_host()
        assert b.set.position == P == a.set.position
    for _, cap_a, _, cap_b, _ in caps:
        cap_a.destroy()
        cap_b.destroy()
    a.set.destroy()
    b.set.destroy()


def test_restore_static_matches_restore_two_calls_in_a_row(esc, ctx):
    # the config-1 layer mix at a reduced size: fold states (fixed rows) + per-token KV rows, 16 segments, one table
    specs = synth.hybrid_layout(512, n_linear=6, n_full=2, H=4, dk=64, dv=64, kv_heads=2, head_dim=64)
    _two_restores_match(esc, ctx, specs, 512, 100, seed=11)


def test_restore_static_several_tables_and_odd_sizes(esc, ctx):
    # 306 segments (three tables of 112), odd sizes and 1-byte tails; then a boundary whose per-token rows are empty
    specs = [synth.RowSpec("robot", 640, 640), synth.RowSpec("odd", 100003, 100003), synth.RowSpec("tok3", 3 * 1000 + 5, 5, 3),
             synth.RowSpec("seg", 300 * 1000, 7, 9, 300, 1000), synth.RowSpec("tile+1", 16385, 16385),
             synth.RowSpec("kv", 2 * 70000, 0, 640, 2, 70000)]
    assert sum(s.n_seg for s in specs) == 306
    _two_restores_match(esc, ctx, specs, 97, 0, seed=12)


def test_restore_static_rejects_what_it_cannot_hold(esc, ctx):
    limit = esc.lib.esc_restore_static_max_segments()
    assert limit == 448
    specs = [synth.RowSpec("many", (limit + 1) * 256, 16, 2, limit + 1, 256)]
    live = LiveSet(esc, ctx, specs, (13,))
    cap, slab = _snapshot(esc, live, 5)
    live.fill(14)
    before = [d.clone() for d in live.dev]
    live.set.set_position(3)
    with pytest.raises(esc.EscError) as ei:
        esc.restore_static(live.set, cap)
    assert ei.value.code == esc.ERR_CAPACITY
    torch.cuda.synchronize()
    assert live.set.position == 3 and all(torch.equal(x, y) for x, y in zip(before, live.dev))   # nothing was enqueued
    esc.restore(live.set, cap)   # the existing path has no such limit
    torch.cuda.synchronize()
    assert live.set.position == 5
    # pairing rules as esc_restore: wrong digest, a capsule of another layout
    with pytest.raises(esc.EscError) as ei:
        esc.restore_static(live.set, cap, expect_prefix_digest=1)
    assert ei.value.code in (esc.ERR_MISMATCH, esc.ERR_CAPACITY)
    other = LiveSet(esc, ctx, [synth.RowSpec("x", 4096, 4096)], (15,))
    with pytest.raises(esc.EscError) as ei:
        esc.restore_static(other.set, cap)
    assert ei.value.code == esc.ERR_MISMATCH
    cap.destroy()
    live.set.destroy()
    other.set.destroy()
