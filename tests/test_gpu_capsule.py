"""-m gpu parity tests of the capsule verbs (snapshot / restore / fork / rollback) through the
C ABI, against the byte-level memcpy oracle.  Bar: bit-exact (integer views).

Test designs follow the paper's own correctness layers: (1) byte restore,
(2) state completeness under adversarially dirtied live buffers, fork branches, rollback,
"raises rather than a partial capsule"."""
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


def _slab(n):
    return torch.empty(n, dtype=torch.uint8, device=DEV)


def _check_snapshot_matches_oracle(live, cap_slab, P):
    rows = live.oracle_rows()
    ref = oracle.capsule_snapshot(rows, P)
    got = cap_slab.cpu().numpy()
    assert got.nbytes >= ref.nbytes
    for r, spec in enumerate(live.specs):
        sv = spec.fixed_bytes + P * spec.bytes_per_token
        for s in range(spec.n_seg):
            off = oracle.capsule_seg_offset(rows, P, r, s)
            assert np.array_equal(got[off:off + sv], ref[off:off + sv]), (spec.name, s)
    return ref


def _small_hybrid(t_max, **kw):
    # the config-1 layer mix (3 linear : 1 full) at a reduced size so the oracle twin stays small
    return synth.hybrid_layout(t_max, n_linear=6, n_full=2, H=4, dk=64, dv=64, kv_heads=2, head_dim=64, **kw)


@pytest.mark.parametrize("head_major", [False, True])
@pytest.mark.parametrize("P", [0, 1, 100, 512])
def test_snapshot_dirty_restore_bit_exact(esc, ctx, head_major, P):
    specs = _small_hybrid(512, head_major=head_major)
    live = LiveSet(esc, ctx, specs, (1, int(head_major), P))
    slab_bytes, payload = live.set.capsule_bytes(P)
    assert slab_bytes == oracle.capsule_slab_bytes(live.oracle_rows(), P)
    assert payload == oracle.capsule_payload_bytes(live.oracle_rows(), P)
    slab = _slab(slab_bytes)
    cap = esc.snapshot(live.set, P, 64 if P % 64 == 0 else 0, slab, prefix_digest=0xABCD)
    torch.cuda.synchronize()
    ref_slab = _check_snapshot_matches_oracle(live, slab, P)
    info = cap.info()
    assert info.boundary == P and info.payload_bytes == payload and info.slab_bytes == slab_bytes
    assert info.prefix_digest == 0xABCD and info.layout_digest == live.set.layout_digest
    assert info.n_rows == len(specs) and info.n_segments == sum(s.n_seg for s in specs)
    # adversarial dirty: an unrelated run's bytes, then 0xFF (NaN patterns) — restore must bring back P's bytes
    for pat in (None, 0xFF):
        live.fill(77, P, pattern=pat)
        esc.restore(live.set, cap, expect_prefix_digest=0xABCD)
        oracle.capsule_restore(live.oracle_rows(), P, ref_slab)   # oracle restores into the same dirtied twin
        live.assert_equals_host()                                  # valid ranges restored, the rest untouched
    assert live.set.position == P
    cap.destroy()
    live.set.destroy()


def test_odd_sizes_and_unaligned_pointers(esc, ctx):
    # the 640-byte robot capsule, 1-byte-granular tails, odd per-token sizes, and
    # buffers whose base is not 16-byte aligned (byte path)
    specs = [synth.RowSpec("robot", 640, 640), synth.RowSpec("one", 1, 1), synth.RowSpec("odd", 100003, 100003),
             synth.RowSpec("tok3", 3 * 1000 + 5, 5, 3), synth.RowSpec("tile+1", 16385, 16385),
             synth.RowSpec("seg", 4 * 1000, 7, 9, 4, 1000)]
    for off in (0, 1, 8):
        live = LiveSet(esc, ctx, specs, (2, off), offset_bytes=off)
        P = 97
        slab = _slab(live.set.capsule_bytes(P)[0])
        cap = esc.snapshot(live.set, P, 0, slab)
        torch.cuda.synchronize()
        ref = _check_snapshot_matches_oracle(live, slab, P)
        live.fill(3, off)
        esc.restore(live.set, cap)
        oracle.capsule_restore(live.oracle_rows(), P, ref)
        live.assert_equals_host()
        cap.destroy()
        live.set.destroy()


def test_fork_then_rollback(esc, ctx):
    # config 3 in miniature: one capsule -> 8 sessions, each dirtied differently, rolled back, byte-identical
    specs = _small_hybrid(1024)
    P = 768
    src = LiveSet(esc, ctx, specs, (3, 0))
    slab = _slab(src.set.capsule_bytes(P)[0])
    cap = esc.snapshot(src.set, P, 64, slab)
    ref = oracle.capsule_snapshot(src.oracle_rows(), P)
    sessions = [LiveSet(esc, ctx, specs, (3, 1 + i)) for i in range(8)]
    esc.fork(cap, [s.set for s in sessions])
    for s in sessions:
        oracle.capsule_restore(s.oracle_rows(), P, ref)
        s.assert_equals_host()
        assert s.set.position == P
    # fork == n restores, byte for byte
    twin = LiveSet(esc, ctx, specs, (3, 1))
    esc.restore(twin.set, cap)
    torch.cuda.synchronize()
    for a, b in zip(twin.dev, sessions[0].dev):
        assert torch.equal(a, b)
    # each session appends 128 tokens (dirties beyond P and the fold states), then rolls back
    for i, s in enumerate(sessions):
        s.fill(99, i)
        s.set.set_position(P + 128)
        esc.rollback(s.set, cap)
        oracle.capsule_restore(s.oracle_rows(), P, ref)
        s.assert_equals_host()
        assert s.set.position == P
    # rollback to a LATER boundary than the session holds is refused
    sessions[0].set.set_position(P - 64)
    with pytest.raises(esc.EscError) as e:
        esc.rollback(sessions[0].set, cap)
    assert e.value.code == esc.ERR_MISMATCH


def test_errors_are_loud_and_enqueue_nothing(esc, ctx):
    specs = _small_hybrid(256)
    live = LiveSet(esc, ctx, specs, (4, 0))
    need = live.set.capsule_bytes(128)[0]
    slab = _slab(need)
    slab.fill_(0x5A)
    with pytest.raises(esc.EscError) as e:   # unaligned boundary
        esc.snapshot(live.set, 100, 64, slab)
    assert e.value.code == esc.ERR_UNALIGNED
    with pytest.raises(esc.EscError) as e:   # beyond capacity
        esc.snapshot(live.set, 257, 0, slab)
    assert e.value.code == esc.ERR_CAPACITY
    with pytest.raises(esc.EscError) as e:   # slab too small
        esc.snapshot(live.set, 128, 64, slab, storage_bytes=need - 1)
    assert e.value.code == esc.ERR_CAPACITY
    torch.cuda.synchronize()
    assert bool((slab == 0x5A).all()), "a failed snapshot wrote into the slab (partial capsule)"
    cap = esc.snapshot(live.set, 100, 64, slab, flags=esc.SNAPSHOT_ALLOW_UNALIGNED)
    assert cap.info().aligned == 0
    cap.destroy()
    cap = esc.snapshot(live.set, 128, 64, slab, prefix_digest=7)
    # wrong prefix digest, wrong layout, too-small live set
    with pytest.raises(esc.EscError) as e:
        esc.restore(live.set, cap, expect_prefix_digest=8)
    assert e.value.code == esc.ERR_MISMATCH
    other = LiveSet(esc, ctx, _small_hybrid(256, head_major=True), (4, 1))
    with pytest.raises(esc.EscError) as e:
        esc.restore(other.set, cap)
    assert e.value.code == esc.ERR_MISMATCH
    small = LiveSet(esc, ctx, _small_hybrid(64), (4, 2))
    before = [d.clone() for d in small.dev]
    with pytest.raises(esc.EscError) as e:
        esc.restore(small.set, cap)
    assert e.value.code == esc.ERR_CAPACITY
    torch.cuda.synchronize()
    for a, b in zip(before, small.dev):
        assert torch.equal(a, b)
    with pytest.raises(esc.EscError):        # a capsule is not a live set
        esc.restore(cap, cap)
    live.set.set_position(64)
    with pytest.raises(esc.EscError) as e:   # live position != P
        esc.snapshot(live.set, 128, 64, slab)
    assert e.value.code == esc.ERR_MISMATCH


def test_table7_shaped_sizes(esc, ctx):
    # bytes(P) = fixed + P * per_token, the form of Table 7; ours: 18 MiB + 24 KiB/token
    specs = synth.hybrid_layout(16384)
    bufs = torch.empty(1, dtype=torch.uint8, device=DEV)   # sizes only: register one dummy address per row
    live = esc.bufset_create(ctx, [(s.name, bufs.data_ptr(), s.capacity_bytes, s.fixed_bytes, s.bytes_per_token,
                                    s.n_seg, s.seg_stride) for s in specs])
    for P in (2048, 4096, 8192, 16384):
        slab_bytes, payload = live.capsule_bytes(P)
        assert payload == 18 * 2**20 + P * 24 * 1024
        assert slab_bytes == payload    # every row is a 256-B multiple: no padding
    live.destroy()


def test_full_size_config1_restore_sampled(esc, ctx):
    # config 1 at full size (66 MiB, 30 segments), the launch configuration bench.py times
    specs = synth.hybrid_layout(2048)
    P = 2048
    live = LiveSet(esc, ctx, specs, (5, 0))
    slab = _slab(live.set.capsule_bytes(P)[0])
    cap = esc.snapshot(live.set, P, 64, slab)
    ref = oracle.capsule_snapshot(live.oracle_rows(), P)
    torch.cuda.synchronize()
    assert np.array_equal(slab.cpu().numpy(), ref)
    live.fill(6, 0)
    esc.restore(live.set, cap)
    oracle.capsule_restore(live.oracle_rows(), P, ref)
    live.assert_equals_host()


@pytest.mark.parametrize("head_major", [False, True])
def test_host_tier_demote_restore_promote_bit_exact(esc, ctx, head_major):
    # SURVEY section 8(f) #2 / PAPER.md:122,125-126,145: tiered handle; promotion = host-backed buffer + async copy.
    # The host-tier slab holds the oracle's bytes; restore / fork straight from it (zero-copy over the host link) and
    # promote back to a device slab are byte-exact.
    P = 448
    specs = _small_hybrid(512, head_major=head_major)
    live = LiveSet(esc, ctx, specs, (5, int(head_major)))
    slab_bytes, payload = live.set.capsule_bytes(P)
    slab = _slab(slab_bytes)
    cap = esc.snapshot(live.set, P, 64, slab, prefix_digest=77)
    host = torch.zeros(slab_bytes, dtype=torch.uint8).pin_memory()
    hcap = esc.capsule_demote(cap, host)
    torch.cuda.synchronize()
    hi = hcap.info()
    assert hi.tier == esc.TIER_HOST and cap.info().tier == esc.TIER_GPU
    assert (hi.boundary, hi.payload_bytes, hi.slab_bytes, hi.prefix_digest, hi.layout_digest) == (
        P, payload, slab_bytes, 77, live.set.layout_digest)
    ref_slab = _check_snapshot_matches_oracle(live, host, P)       # host slab == oracle's memcpy capsule on valid ranges
    slab.fill_(0xEE)                                                # the device slab may go away: the host tier is self-contained
    # restore directly from the host tier after an adversarial dirty
    live.fill(78, 0, pattern=0xFF)
    esc.restore(live.set, hcap, expect_prefix_digest=77)
    oracle.capsule_restore(live.oracle_rows(), P, ref_slab)
    live.assert_equals_host()
    assert live.set.position == P
    # fork from the host tier
    sessions = [LiveSet(esc, ctx, specs, (5, 10 + i)) for i in range(3)]
    esc.fork(hcap, [s.set for s in sessions])
    for s in sessions:
        oracle.capsule_restore(s.oracle_rows(), P, ref_slab)
        s.assert_equals_host()
    # promote into a fresh device slab: a GPU-tier capsule with the same bytes
    slab2 = _slab(slab_bytes)
    cap2 = esc.capsule_promote(hcap, slab2)
    torch.cuda.synchronize()
    assert cap2.info().tier == esc.TIER_GPU
    _check_snapshot_matches_oracle(live, slab2, P)
    live.fill(79, 0)
    esc.rollback(live.set, cap2)
    oracle.capsule_restore(live.oracle_rows(), P, ref_slab)
    live.assert_equals_host()
    # errors: pageable host memory, wrong tier, short storage — nothing enqueued, no handle returned
    with pytest.raises(esc.EscError) as e:
        esc.capsule_demote(cap, torch.zeros(slab_bytes + 256, dtype=torch.uint8)[: slab_bytes])
    assert e.value.code in (esc.ERR_INVALID, esc.ERR_UNALIGNED)
    with pytest.raises(esc.EscError) as e:
        esc.capsule_demote(hcap, host)
    assert e.value.code == esc.ERR_INVALID
    with pytest.raises(esc.EscError) as e:
        esc.capsule_promote(cap, slab2)
    assert e.value.code == esc.ERR_INVALID
    with pytest.raises(esc.EscError) as e:
        esc.capsule_promote(hcap, slab2[: slab_bytes - 256])
    assert e.value.code == esc.ERR_CAPACITY
    for c in (cap, hcap, cap2):
        c.destroy()


def test_host_tier_capsule_in_graph(esc, ctx):
    # the captured restore node reads whatever capsule is bound: binding a HOST-tier capsule needs no recapture either
    P = 256
    specs = _small_hybrid(512)
    live = LiveSet(esc, ctx, specs, (6, 0))
    slab = _slab(live.set.capsule_bytes(P)[0])
    cap = esc.snapshot(live.set, P, 64, slab)
    host = torch.zeros(slab.numel(), dtype=torch.uint8).pin_memory()
    hcap = esc.capsule_demote(cap, host)
    torch.cuda.synchronize()
    ref = oracle.capsule_snapshot(live.oracle_rows(), P)
    stream = torch.cuda.Stream()
    graph = esc.graph_capture(ctx, live.set, P, [], stream)
    for c in (cap, hcap, cap):
        live.fill(80, 0, pattern=0xFF)
        torch.cuda.synchronize()
        graph.set_capsule(c, stream)
        graph.launch(stream)
        stream.synchronize()
        oracle.capsule_restore(live.oracle_rows(), P, ref)
        live.assert_equals_host()
    graph.destroy()


def test_seeded_layout_fuzz_bit_exact(esc, ctx):
    # 12 seeded random buffer sets (odd sizes, mixed fixed / per-token rows, multi-segment rows, unaligned base offsets):
    # snapshot -> dirty -> restore and a 3-way fork, byte-exact against the memcpy oracle
    rng = np.random.default_rng(20538)
    for it in range(12):
        specs = []
        t_max = int(rng.integers(8, 200))
        for r in range(int(rng.integers(1, 9))):
            kind = int(rng.integers(0, 3))
            if kind == 0:
                nb = int(rng.integers(1, 5000))
                specs.append(synth.RowSpec("r%02d.fixed" % r, nb, nb, 0, 1, 0))
            elif kind == 1:
                bpt = int(rng.integers(1, 300))
                specs.append(synth.RowSpec("r%02d.tok" % r, t_max * bpt, 0, bpt, 1, 0))
            else:
                bpt, nseg = int(rng.integers(1, 120)), int(rng.integers(2, 5))
                stride = t_max * bpt + int(rng.integers(0, 40))
                specs.append(synth.RowSpec("r%02d.seg" % r, stride * nseg, 0, bpt, nseg, stride))
        P = int(rng.integers(0, t_max + 1))
        live = LiveSet(esc, ctx, specs, (30, it), offset_bytes=int(rng.choice([0, 0, 1, 3, 16])))
        slab = _slab(live.set.capsule_bytes(P)[0] + 256)
        cap = esc.snapshot(live.set, P, 0, slab)
        torch.cuda.synchronize()
        ref = _check_snapshot_matches_oracle(live, slab, P)
        live.fill(31, it, pattern=0xFF)
        esc.restore(live.set, cap)
        oracle.capsule_restore(live.oracle_rows(), P, ref)
        live.assert_equals_host()
        forks = [LiveSet(esc, ctx, specs, (32, it, f), offset_bytes=int(rng.choice([0, 2]))) for f in range(3)]
        esc.fork(cap, [f.set for f in forks])
        for f in forks:
            oracle.capsule_restore(f.oracle_rows(), P, ref)
            f.assert_equals_host()
        cap.destroy()
