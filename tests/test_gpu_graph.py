"""-m gpu tests of the captured replay plan: restore + 18-layer suffix scan as ONE CUDA graph
(BASELINE config 1), capsule swapped between replays without recapture."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_20537_b200 import synth
from gpu_util import (to_dev, DEV, TOL_O, TOL_S, LiveSet, assert_state_close, bits_equal, err_o, err_s, esc_mod, sample_heads,
                      scan_dev_inputs)

pytestmark = pytest.mark.gpu

B, H, DK, DV, CHUNK, SUFFIX = 1, 16, 128, 128, 64, 64


@pytest.fixture(scope="module")
def esc():
    return esc_mod()


@pytest.fixture(scope="module")
def ctx(esc):
    c = esc.Ctx(0)
    yield c
    c.close()


def _hybrid_live(esc, ctx, t_max, seed):
    specs = synth.hybrid_layout(t_max)
    live = LiveSet(esc, ctx, specs, (20, seed))
    lin = [i for i, s in enumerate(specs) if ".lin." in s.name]
    for n, i in enumerate(lin):   # fold states must be finite floats, not random bytes
        live.set_row(i, synth.scan_state(B, H, DK, DV, seed_ids=(20, seed, n), scale=0.3))
    return live, lin


def test_restore_plus_suffix_scan_graph(esc, ctx):
    P = 2048
    live, lin = _hybrid_live(esc, ctx, P + SUFFIX, 0)
    states = [live.dev[i].view(torch.float32).view(B, H, DK, DV) for i in lin]
    key = esc.shape_key_make(B, H, DK, DV, esc.DTYPE_BF16, esc.DTYPE_F32, CHUNK)
    ins = [synth.scan_inputs(B, SUFFIX, H, DK, DV, seed_ids=(21, n)) for n in range(len(lin))]
    dev_ins = [scan_dev_inputs(si) for si in ins]
    outs = [torch.zeros((B, SUFFIX, H, DV), dtype=torch.float32, device=DEV) for _ in lin]

    # two capsules with different contents (A: the initial live set; B: another prefill's bytes)
    slab_a = torch.empty(live.set.capsule_bytes(P)[0], dtype=torch.uint8, device=DEV)
    cap_a = esc.snapshot(live.set, P, CHUNK, slab_a)
    s0_a = [s.clone() for s in states]
    live.fill(22, 0)
    for n, i in enumerate(lin):
        live.set_row(i, synth.scan_state(B, H, DK, DV, seed_ids=(22, n), scale=0.3))
    slab_b = torch.empty_like(slab_a)
    cap_b = esc.snapshot(live.set, P, CHUNK, slab_b)
    torch.cuda.synchronize()

    def by_verbs(cap):
        esc.restore(live.set, cap)
        for n in range(len(lin)):
            q, k, v, g = dev_ins[n]
            esc.linattn_scan(ctx, key, q, k, v, g, states[n], states[n], outs[n], SUFFIX, SUFFIX, CHUNK)
        torch.cuda.synchronize()
        return [o.clone() for o in outs], [d.clone() for d in live.dev]

    exp_a = by_verbs(cap_a)
    exp_b = by_verbs(cap_b)
    assert not bits_equal(exp_a[0][0], exp_b[0][0])

    stream = torch.cuda.Stream()
    layers = [esc.scan_args(key, *dev_ins[n], states[n], states[n], outs[n], SUFFIX, SUFFIX, CHUNK)
              for n in range(len(lin))]
    graph = esc.graph_capture(ctx, live.set, P, layers, stream)
    with pytest.raises(esc.EscError):          # no capsule bound yet
        graph.launch(stream)
    for cap, (exp_o, exp_live) in ((cap_a, exp_a), (cap_b, exp_b), (cap_a, exp_a)):
        live.fill(23, 0, pattern=0xFF)         # dirty every live buffer (NaN patterns)
        for o in outs:
            o.fill_(float("nan"))
        torch.cuda.synchronize()
        graph.set_capsule(cap, stream)         # swap the capsule: no recapture
        graph.launch(stream)
        stream.synchronize()
        for o, e in zip(outs, exp_o):
            assert bits_equal(o, e)
        # live buffers: fold states advanced by the suffix, KV valid ranges restored; beyond-valid stays dirty
        for i, (d, e) in enumerate(zip(live.dev, exp_live)):
            sv = live.specs[i].fixed_bytes + P * live.specs[i].bytes_per_token
            assert torch.equal(d[:sv], e[:sv]), live.specs[i].name
            assert bool((d[sv:] == 0xFF).all())
        assert live.set.position == P

    # the graph's result against the oracle for one layer (state_in = capsule A's fold state)
    q, k, v, g = ins[3].as_f32()
    o_ref, s_ref = oracle.linattn_recurrence(q, k, v, g, s0_a[3].cpu().numpy().astype(np.float64))
    assert err_o(outs[3].cpu().numpy(), o_ref) <= TOL_O
    assert_state_close(states[3], s_ref)
    graph.destroy()


def test_delta_rule_layers_in_a_captured_plan(esc, ctx):
    """esc_scan_args.kind = ESC_SCAN_GDN: the restore node followed by one gated delta-rule scan per layer (the recurrence of the
    paper's own model family) replayed as ONE graph; bit-identical to restore + esc_gdn_scan calls, capsule
    swapped without recapture, a mixed plan (delta-rule and linear-attention layers) accepted, one layer against the oracle."""
    P = 2048
    live, lin = _hybrid_live(esc, ctx, P + SUFFIX, 5)
    states = [live.dev[i].view(torch.float32).view(B, H, DK, DV) for i in lin]
    key = esc.shape_key_make(B, H, DK, DV, esc.DTYPE_BF16, esc.DTYPE_F32, CHUNK)
    ins = [synth.scan_inputs(B, SUFFIX, H, DK, DV, seed_ids=(61, n), gate="slow") for n in range(len(lin))]
    betas = [synth.gdn_beta(B, SUFFIX, H, seed_ids=(61, n)) for n in range(len(lin))]
    dev_ins = [scan_dev_inputs(si) for si in ins]
    dev_betas = [to_dev(b_) for b_ in betas]
    outs = [torch.zeros((B, SUFFIX, H, DV), dtype=torch.float32, device=DEV) for _ in lin]
    for n, i in enumerate(lin):
        live.set_row(i, synth.scan_state(B, H, DK, DV, seed_ids=(62, n), scale=0.3))
    slab_a = torch.empty(live.set.capsule_bytes(P)[0], dtype=torch.uint8, device=DEV)
    cap_a = esc.snapshot(live.set, P, CHUNK, slab_a)
    s0_a = [s.clone() for s in states]
    for n, i in enumerate(lin):
        live.set_row(i, synth.scan_state(B, H, DK, DV, seed_ids=(63, n), scale=0.3))
    slab_b = torch.empty_like(slab_a)
    cap_b = esc.snapshot(live.set, P, CHUNK, slab_b)
    torch.cuda.synchronize()
    gdn_layer = lambda n: n % 3 != 2   # a mixed plan: every third layer is a linear-attention layer

    def by_verbs(cap):
        esc.restore(live.set, cap)
        for n in range(len(lin)):
            q, k, v, g = dev_ins[n]
            if gdn_layer(n):
                esc.gdn_scan(ctx, key, q, k, v, g, dev_betas[n], states[n], states[n], outs[n], SUFFIX, SUFFIX)
            else:
                esc.linattn_scan(ctx, key, q, k, v, g, states[n], states[n], outs[n], SUFFIX, SUFFIX, CHUNK)
        torch.cuda.synchronize()
        return [o.clone() for o in outs], [s.clone() for s in states]

    exp_a, exp_b = by_verbs(cap_a), by_verbs(cap_b)
    assert not bits_equal(exp_a[0][0], exp_b[0][0])
    stream = torch.cuda.Stream()
    layers = [esc.scan_args(key, *dev_ins[n], states[n], states[n], outs[n], SUFFIX, SUFFIX, CHUNK,
                            beta=dev_betas[n] if gdn_layer(n) else None) for n in range(len(lin))]
    graph = esc.graph_capture(ctx, live.set, P, layers, stream)
    for cap, (exp_o, exp_s) in ((cap_a, exp_a), (cap_b, exp_b), (cap_a, exp_a)):
        for o in outs:
            o.fill_(float("nan"))
        for s_ in states:
            s_.fill_(float("nan"))
        torch.cuda.synchronize()
        graph.set_capsule(cap, stream)
        graph.launch(stream)
        stream.synchronize()
        for n in range(len(lin)):
            assert bits_equal(outs[n], exp_o[n]) and bits_equal(states[n], exp_s[n]), n
    q, k, v, g = ins[0].as_f32()
    o_ref, s_ref = oracle.gdn_recurrence(q, k, v, g, betas[0], s0_a[0].cpu().numpy().astype(np.float64))
    assert err_o(outs[0].cpu().numpy(), o_ref) <= TOL_O
    assert_state_close(states[0], s_ref)
    graph.destroy()
    # argument contract: beta on a linear-attention layer, a delta-rule layer without beta, an unknown kind
    bad = esc.scan_args(key, *dev_ins[0], states[0], states[0], outs[0], SUFFIX, SUFFIX, CHUNK)
    bad.beta = dev_betas[0].data_ptr()
    with pytest.raises(esc.EscError):
        esc.graph_capture(ctx, None, 0, [bad], stream)
    bad = esc.scan_args(key, *dev_ins[0], states[0], states[0], outs[0], SUFFIX, SUFFIX, CHUNK, beta=dev_betas[0])
    bad.beta = None
    with pytest.raises(esc.EscError):
        esc.graph_capture(ctx, None, 0, [bad], stream)
    bad = esc.scan_args(key, *dev_ins[0], states[0], states[0], outs[0], SUFFIX, SUFFIX, CHUNK)
    bad.kind = 7
    with pytest.raises(esc.EscError):
        esc.graph_capture(ctx, None, 0, [bad], stream)
    cap_a.destroy()
    cap_b.destroy()
    live.set.destroy()


def test_cold_plan_graph_matches_direct_calls(esc, ctx):
    # a plan without a restore node: n layers of cold scans in one launch
    T, n_layers = 512, 3
    key = esc.shape_key_make(B, H, DK, DV, esc.DTYPE_BF16, esc.DTYPE_F32, CHUNK)
    dev_ins = [scan_dev_inputs(synth.scan_inputs(B, T, H, DK, DV, seed_ids=(24, n))) for n in range(n_layers)]
    st = [torch.empty((B, H, DK, DV), dtype=torch.float32, device=DEV) for _ in range(n_layers)]
    outs = [torch.empty((B, T, H, DV), dtype=torch.float32, device=DEV) for _ in range(n_layers)]
    for n in range(n_layers):
        esc.linattn_scan(ctx, key, *dev_ins[n], None, st[n], outs[n], T, T, CHUNK)
    torch.cuda.synchronize()
    exp = [(o.clone(), s.clone()) for o, s in zip(outs, st)]
    stream = torch.cuda.Stream()
    graph = esc.graph_capture(ctx, None, 0, [esc.scan_args(key, *dev_ins[n], None, st[n], outs[n], T, T, CHUNK)
                                             for n in range(n_layers)], stream)
    for o, s in zip(outs, st):
        o.fill_(float("nan"))
        s.fill_(float("nan"))
    torch.cuda.synchronize()
    graph.launch(stream)
    stream.synchronize()
    for (eo, es_), o, s in zip(exp, outs, st):
        assert bits_equal(o, eo) and bits_equal(s, es_)
    graph.destroy()


def test_config3_fork_continue_rollback_replay(esc, ctx):
    # BASELINE config 3: one 8k-prefix capsule of the 24-layer hybrid layout forked into 8 sessions in device memory, each
    # continued with 128 distinct seeded suffix tokens, then rolled back to the capsule and replayed: states, outputs and
    # the capsule's valid ranges byte-identical to the first pass.
    from paper_2606_20537_b200 import workload
    P, n_sess, suffix = 8192, 8, 128
    key = esc.shape_key_make(B, H, DK, DV, esc.DTYPE_BF16, esc.DTYPE_F32, CHUNK)
    src = workload.HybridSession(ctx, P + suffix, seed=40, device=DEV)
    slab = src.new_slab(P)
    src.set.set_position(P)
    cap = esc.snapshot(src.set, P, CHUNK, slab)
    assert cap.info().payload_bytes == 18 * (1 << 20) + 24576 * P      # 210 MiB
    sessions = [workload.HybridSession(ctx, P + suffix, seed=41 + i, device=DEV) for i in range(n_sess)]
    inputs = [workload.SuffixInputs(len(src.lin), suffix, seed=60 + i, device=DEV) for i in range(n_sess)]
    esc.fork(cap, [s.set for s in sessions])
    torch.cuda.synchronize()
    for s in sessions:            # every session's valid ranges == the source's, byte for byte
        for spec, a, b_ in zip(s.specs, s.bufs, src.bufs):
            nv = spec.fixed_bytes + P * spec.bytes_per_token
            assert torch.equal(a.view(torch.uint8).view(-1)[:nv], b_.view(torch.uint8).view(-1)[:nv]), spec.name

    def continue_all():
        res = []
        for s, inp in zip(sessions, inputs):
            for n in range(len(s.lin)):
                q, k, v, g = inp.dev[n]
                esc.linattn_scan(ctx, key, q, k, v, g, s.states[n], s.states[n], inp.out[n], suffix, suffix, CHUNK)
            # the harness "appends" 128 KV tokens: dirties [P, P+128) of every KV row
            for spec, buf in zip(s.specs, s.bufs):
                if spec.bytes_per_token:
                    buf.view(torch.uint8).view(-1)[P * spec.bytes_per_token:(P + suffix) * spec.bytes_per_token].fill_(0x5A)
            s.set.set_position(P + suffix)
        torch.cuda.synchronize()
        for s, inp in zip(sessions, inputs):
            res.append(([st.clone() for st in s.states], inp.out_dev.clone()))
        return res

    first = continue_all()
    assert not bits_equal(first[0][0][0], first[1][0][0])            # distinct suffixes: the branches differ
    for s in sessions:
        esc.rollback(s.set, cap)
        assert s.set.position == P
    torch.cuda.synchronize()
    for s in sessions:
        for n, st in enumerate(s.states):
            assert bits_equal(st, src.states[n])
    for inp in inputs:
        inp.out_dev.fill_(0xFF)
    second = continue_all()
    for (st1, o1), (st2, o2) in zip(first, second):
        assert torch.equal(o1, o2)
        for a, b_ in zip(st1, st2):
            assert bits_equal(a, b_)
    # one branch against the oracle (state_in = the capsule's fold state)
    si = synth.scan_inputs(B, suffix, H, DK, DV, seed_ids=(31, 60 + 3, 5))
    qf, kf, vf, gf = si.as_f32()
    o_ref, s_ref = oracle.linattn_recurrence(qf, kf, vf, gf, src.states[5].cpu().numpy().astype(np.float64))
    assert err_o(inputs[3].out[5].cpu().numpy(), o_ref) <= TOL_O
    assert_state_close(second[3][0][5], s_ref)


def test_config2_capsule_and_warm_graph_equal_cold_graph(esc, ctx):
    # BASELINE config 2 end to end at full size (PAPER.md:165 three correctness layers, :223 "chunk-aligned long boundary =
    # cold full prefill", :243-252 the 16k row of Table 7):
    #   (1) the 402 MiB capsule at P = 16384: snapshot / restore byte-exact against the memcpy oracle;
    #   (2) ONE graph [restore(16384) + 18 x scan(64)] after an adversarial dirty is bit-identical to the cold graph
    #       [18 x scan(16448)] on o[16384:16448] and on all 18 final states;
    #   (3) one layer against the fp64 oracle on a seeded sample of heads.
    P, T = 16384, 16384 + SUFFIX
    live, lin = _hybrid_live(esc, ctx, T, 7)
    n_lin = len(lin)
    assert n_lin == 18
    states = [live.dev[i].view(torch.float32).view(B, H, DK, DV) for i in lin]
    key = esc.shape_key_make(B, H, DK, DV, esc.DTYPE_BF16, esc.DTYPE_F32, CHUNK)
    # per-layer inputs: three seeded draws, rolled along T for the other layers (same distribution, distinct per layer)
    base = [synth.scan_inputs(B, T, H, DK, DV, seed_ids=(25, n)) for n in range(3)]
    base_dev = [scan_dev_inputs(si) for si in base]
    shift = lambda n: 0 if n < 3 else 64 * 7 * n       # a multiple of the chunk: the rolled layers stay chunk-aligned
    dev_ins = [tuple(torch.roll(t, shifts=shift(n), dims=1) for t in base_dev[n % 3]) for n in range(n_lin)]
    stream = torch.cuda.Stream()

    # ---- cold: 18 x scan(16448) from S_0 = 0 as one graph (the configuration bench.py's warm_vs_cold times) ----
    s_cold = [torch.full((B, H, DK, DV), float("nan"), dtype=torch.float32, device=DEV) for _ in range(n_lin)]
    o_cold = [torch.full((B, T, H, DV), float("nan"), dtype=torch.float32, device=DEV) for _ in range(n_lin)]
    cold = esc.graph_capture(ctx, None, 0, [esc.scan_args(key, *dev_ins[n], None, s_cold[n], o_cold[n], T, T, CHUNK)
                                            for n in range(n_lin)], stream)
    torch.cuda.synchronize()      # the inputs and the NaN fills were enqueued on the default stream; `stream` does not wait for it
    cold.launch(stream)
    stream.synchronize()
    cold.destroy()
    o_cold_tail = [o[:, P:].clone() for o in o_cold]

    # ---- prefill to P in the live fold states (S_0 = 0), snapshot: the 402 MiB capsule ----
    for n in range(n_lin):
        q, k, v, g = dev_ins[n]
        esc.linattn_scan(ctx, key, q, k, v, g, None, states[n], o_cold[n], P, T, CHUNK)   # o[:P] rewritten with the same bits
    torch.cuda.synchronize()
    for n, i in enumerate(lin):                               # host twin of the fold states for the memcpy oracle
        live.host[i][:] = live.dev[i].cpu().numpy()
    live.set.set_position(P)
    slab_bytes, payload = live.set.capsule_bytes(P)
    assert payload == 18 * (1 << 20) + 24576 * P == 421527552      # 402 MiB
    slab = torch.empty(slab_bytes, dtype=torch.uint8, device=DEV)
    cap = esc.snapshot(live.set, P, CHUNK, slab)
    torch.cuda.synchronize()
    ref = oracle.capsule_snapshot(live.oracle_rows(), P)
    assert np.array_equal(slab.cpu().numpy(), ref), "402 MiB capsule differs from the oracle's memcpy capsule"
    # restore by the verb after an adversarial dirty: byte-exact on every row, beyond-valid bytes keep the dirt
    live.fill(26, 0, pattern=0xFF)
    esc.restore(live.set, cap)
    oracle.capsule_restore(live.oracle_rows(), P, ref)
    live.assert_equals_host()

    # ---- warm: ONE graph [restore(16384) + 18 x scan(64)] ----
    o_warm = [torch.full((B, SUFFIX, H, DV), float("nan"), dtype=torch.float32, device=DEV) for _ in range(n_lin)]
    layers = []
    for n in range(n_lin):
        q, k, v, g = dev_ins[n]
        layers.append(esc.scan_args(key, q[:, P:], k[:, P:], v[:, P:], g[:, P:], states[n], states[n], o_warm[n],
                                    SUFFIX, T, CHUNK))
    warm = esc.graph_capture(ctx, live.set, P, layers, stream)
    live.fill(27, 0, pattern=0xFF)
    torch.cuda.synchronize()
    warm.set_capsule(cap, stream)
    warm.launch(stream)
    stream.synchronize()
    for n in range(n_lin):
        assert bits_equal(o_warm[n], o_cold_tail[n]), "layer %d: warm o[16384:] differs from the cold graph" % n
        assert bits_equal(states[n], s_cold[n]), "layer %d: warm S_16448 differs from the cold graph" % n
    # KV rows: valid ranges restored byte-exactly (the oracle's memcpy twin), beyond-valid bytes still dirty
    oracle.capsule_restore(live.oracle_rows(), P, ref)
    for i, spec in enumerate(live.specs):
        if spec.bytes_per_token:
            assert np.array_equal(live.dev[i].cpu().numpy(), live.host[i]), spec.name
    warm.destroy()
    cap.destroy()

    # ---- one layer against the oracle (seeded sample of heads, whole 16448-token sequence) ----
    n = 1
    q, k, v, g = base[n].as_f32()
    for (b, h) in sample_heads(B, H, 3, 25):
        sl = (slice(b, b + 1), slice(None), slice(h, h + 1))
        o_ref, s_ref = oracle.linattn_recurrence(q[sl], k[sl], v[sl], g[sl])
        assert err_o(o_warm[n][b:b + 1, :, h:h + 1].cpu().numpy(), o_ref[:, P:]) <= TOL_O
        assert err_o(o_cold[n][b:b + 1, :, h:h + 1].cpu().numpy(), o_ref) <= TOL_O
        assert_state_close(states[n][b:b + 1, h:h + 1], s_ref)


def test_plan_table_lru_and_padded_bucket(esc):
    # SURVEY 8(f) #4 / PAPER.md:195,386: bounded Graph[key] table with LRU eviction; a plan captured for a suffix bucket
    # serves a shorter suffix padded with k = v = 0, g = 1 tokens, bit-identically to the unpadded scan.
    ctx = esc.Ctx(0)
    stream = torch.cuda.Stream()
    b_, h_, chunk = 1, 2, 64
    key = esc.shape_key_make(b_, h_, DK, DV, esc.DTYPE_BF16, esc.DTYPE_F32, chunk)
    T = 100
    bucket = esc.suffix_bucket(T, chunk)
    assert bucket == 128
    si = synth.scan_inputs(b_, T, h_, DK, DV, seed_ids=(50,), gate="slow")
    q, k, v, g = scan_dev_inputs(si)
    pad = lambda x, val: torch.cat([x, torch.full((b_, bucket - T) + tuple(x.shape[2:]), val, dtype=x.dtype, device=DEV)], dim=1).contiguous()
    qp, kp, vp, gp = pad(q, 1.0), pad(k, 0.0), pad(v, 0.0), pad(g, 1.0)
    s0 = torch.from_numpy(synth.scan_state(b_, h_, DK, DV, seed_ids=(51,), scale=0.3)).to(DEV)
    # reference: the unpadded T-token scan
    s_ref, o_ref = s0.clone(), torch.zeros((b_, T, h_, DV), dtype=torch.float32, device=DEV)
    esc.linattn_scan(ctx, key, q, k, v, g, s_ref, s_ref, o_ref, T, T, chunk)
    state = s0.clone()
    o = torch.zeros((b_, bucket, h_, DV), dtype=torch.float32, device=DEV)

    def capture(n):
        return esc.graph_capture(ctx, None, 0, [esc.scan_args(key, qp, kp, vp, gp, state, state, o, bucket, bucket, chunk)] * n, stream)

    ctx.plan_table_set_capacity(2)
    pk = [esc.plan_key_make(key, bucket, 0, n) for n in (1, 2, 3)]
    assert ctx.plan_get(pk[0]) is None                       # a new shape needing capture
    g0, g1 = capture(1), capture(2)
    ctx.plan_put(pk[0], g0)
    ctx.plan_put(pk[1], g1)
    # ownership: a plan the table holds cannot be destroyed by the caller, nor be put under a second key
    assert esc.lib.esc_graph_destroy(g0.h) == esc.ERR_INVALID
    with pytest.raises(esc.EscError) as e:
        ctx.plan_put(pk[2], g0)
    assert e.value.code == esc.ERR_INVALID
    plan = ctx.plan_get(pk[0])                               # hit; pk[0] becomes most recently used
    assert plan is not None
    torch.cuda.synchronize()                                 # default-stream set-up before the side stream's launch
    plan.launch(stream)
    stream.synchronize()
    assert bits_equal(o[:, :T], o_ref) and bits_equal(state, s_ref)
    ctx.plan_put(pk[2], capture(3))                          # table full: evicts the least recently used = pk[1]
    assert ctx.plan_get(pk[1]) is None and ctx.plan_get(pk[0]) is not None and ctx.plan_get(pk[2]) is not None
    with pytest.raises(esc.EscError):                        # the evicted plan's wrapper is dead, not dangling
        g1.launch(stream)
    st = ctx.plan_stats()
    assert st == {"size": 2, "hits": 3, "misses": 2, "evictions": 1}
    ctx.plan_table_set_capacity(1)                           # shrinking evicts down to the most recently used (pk[2])
    assert ctx.plan_get(pk[0]) is None and ctx.plan_get(pk[2]) is not None
    assert ctx.plan_stats()["evictions"] == 2
    ctx.close()                                              # the context destroys the plans it still owns


def test_graph_scratch_and_capacity_contract(esc, ctx):
    # include/esc.h "Ownership": the restore node's descriptor table lives in CALLER-owned scratch; a capsule later than the
    # plan's max_boundary is refused; every error is reported before anything is enqueued.
    specs = synth.hybrid_layout(256, n_linear=2, n_full=1, H=2, dk=64, dv=64, kv_heads=1, head_dim=64)
    live = LiveSet(esc, ctx, specs, (90, 0))
    stream = torch.cuda.Stream()
    need = esc.graph_scratch_bytes()
    assert 0 < need <= 8192

    def raw_capture(scratch_ptr, nbytes):
        h = esc._P()
        arr = (esc.ScanArgs * 1)()
        return esc.lib.esc_graph_capture(ctx.h, live.set.h, 128, arr, 0, scratch_ptr, nbytes, stream.cuda_stream, esc.C.byref(h))

    big = torch.zeros(need + 64, dtype=torch.uint8, device=DEV)
    assert raw_capture(None, 0) == esc.ERR_INVALID
    assert raw_capture(big.data_ptr(), need - 1) == esc.ERR_CAPACITY
    assert raw_capture(big.data_ptr() + 4, need) == esc.ERR_UNALIGNED
    scratch = torch.full((need,), 0xAB, dtype=torch.uint8, device=DEV)    # garbage in the scratch must not matter
    graph = esc.graph_capture(ctx, live.set, 128, [], stream, scratch=scratch)
    slab = torch.empty(live.set.capsule_bytes(192)[0], dtype=torch.uint8, device=DEV)
    torch.cuda.synchronize()
    cap_late = esc.snapshot(live.set, 192, 64, slab, stream=stream)
    with pytest.raises(esc.EscError) as e:
        graph.set_capsule(cap_late, stream)                  # boundary 192 > max_boundary 128
    assert e.value.code == esc.ERR_CAPACITY
    cap = esc.snapshot(live.set, 128, 64, slab, stream=stream)
    stream.synchronize()
    ref = oracle.capsule_snapshot(live.oracle_rows(), 128)
    live.fill(91, 0, pattern=0xFF)
    torch.cuda.synchronize()
    graph.set_capsule(cap, stream)
    graph.launch(stream)
    stream.synchronize()
    oracle.capsule_restore(live.oracle_rows(), 128, ref)
    live.assert_equals_host()
    graph.destroy()
