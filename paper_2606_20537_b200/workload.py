"""The hybrid-model workload of BASELINE.json configs 1-3 on the GPU: a 24-layer live buffer set
(18 linear-attention fold states + 6 full-attention layers' K and V buffers), capsule slabs, and the
per-layer suffix-scan inputs.  Plumbing for bench.py / smoke() / tests: torch allocations + seeded
inputs from `synth` + calls into the C ABI (`esc`).  No method arithmetic lives here.
"""
import numpy as np
import torch

from . import esc, synth

B, H, DK, DV = 1, 16, 128, 128


def _bf16_dev(bits: np.ndarray, device):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(device).view(torch.bfloat16)


class HybridSession:
    """One session's live buffer set at capacity `t_max` tokens, registered with the library."""

    def __init__(self, ctx, t_max, seed=0, device="cuda:0", head_major=False):
        self.ctx, self.t_max, self.device = ctx, t_max, device
        self.specs = synth.hybrid_layout(t_max, head_major=head_major)
        self.bufs = []
        self.lin = []       # indices of the fold-state rows
        g = torch.Generator(device=device)
        for i, s in enumerate(self.specs):
            if ".lin." in s.name:
                st = synth.scan_state(B, H, DK, DV, seed_ids=(30, seed, i), scale=0.3)
                t = torch.from_numpy(st).to(device)
                self.lin.append(i)
            else:
                # KV content only matters for byte equality: seeded device-side bf16 N(0,1)
                g.manual_seed(synth.BASE_SEED * 1000 + seed * 100 + i)
                t = torch.randn(s.capacity_bytes // 2, generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)
            self.bufs.append(t)
        self.set = esc.bufset_create(ctx, [(s.name, t, s.capacity_bytes, s.fixed_bytes, s.bytes_per_token, s.n_seg,
                                            s.seg_stride) for s, t in zip(self.specs, self.bufs)])
        self.states = [self.bufs[i].view(B, H, DK, DV) for i in self.lin]

    def capsule_bytes(self, P):
        return self.set.capsule_bytes(P)

    def new_slab(self, P):
        return torch.empty(self.capsule_bytes(P)[0], dtype=torch.uint8, device=self.device)

    def dirty(self, value=float("nan")):
        for t in self.bufs:
            t.fill_(value)


class SuffixInputs:
    """Per-layer q,k,v,g for `T` tokens and the per-layer outputs.  All layers' inputs live in ONE device blob
    (and one pinned host blob), all outputs in another, so an end-to-end step is one H2D and one D2H copy."""

    def __init__(self, n_layers, T, seed=0, device="cuda:0", out_dtype=torch.float32, distinct=True, pinned=False):
        self.T, self.n_layers = T, n_layers
        esz = {torch.float32: 4, torch.bfloat16: 2}[out_dtype]
        nq, nv, ng, no = B * T * H * DK * 2, B * T * H * DV * 2, B * T * H * 4, B * T * H * DV * esz
        al = lambda x: (x + 255) // 256 * 256
        per_layer = 2 * al(nq) + al(nv) + al(ng)
        self.in_dev = torch.empty(n_layers * per_layer, dtype=torch.uint8, device=device)
        self.out_dev = torch.empty(n_layers * al(no), dtype=torch.uint8, device=device)
        self.in_host = torch.empty(n_layers * per_layer, dtype=torch.uint8, pin_memory=True) if pinned else None
        self.out_host = torch.empty(n_layers * al(no), dtype=torch.uint8, pin_memory=True) if pinned else None
        self.dev, self.out = [], []
        first = None
        for n in range(n_layers):
            base = n * per_layer
            offs = [base, base + al(nq), base + 2 * al(nq), base + 2 * al(nq) + al(nv)]
            views = [self.in_dev[offs[0]:offs[0] + nq].view(torch.bfloat16).view(B, T, H, DK),
                     self.in_dev[offs[1]:offs[1] + nq].view(torch.bfloat16).view(B, T, H, DK),
                     self.in_dev[offs[2]:offs[2] + nv].view(torch.bfloat16).view(B, T, H, DV),
                     self.in_dev[offs[3]:offs[3] + ng].view(torch.float32).view(B, T, H)]
            if distinct or first is None:
                si = synth.scan_inputs(B, T, H, DK, DV, seed_ids=(31, seed, n))
                srcs = [si.q_bits, si.k_bits, si.v_bits, si.g]
                for v_, a, o_ in zip(views, srcs, offs):
                    hb = torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1))
                    if self.in_host is not None:
                        self.in_host[o_:o_ + hb.numel()].copy_(hb)
                    v_.view(torch.uint8).view(-1).copy_(hb)
                first = views
            else:
                # same distribution, rolled along T by a layer-dependent shift (cheap for very long T)
                for v_, f_ in zip(views, first):
                    v_.copy_(torch.roll(f_, shifts=17 * n, dims=1))
            self.dev.append(views)
            oo = n * al(no)
            self.out.append(self.out_dev[oo:oo + no].view(out_dtype).view(B, T, H, DV))

    def h2d(self, stream=None):
        self.in_dev.copy_(self.in_host, non_blocking=True)

    def d2h(self, stream=None):
        self.out_host.copy_(self.out_dev, non_blocking=True)

    def h2d_bytes(self):
        return self.in_dev.numel()

    def d2h_bytes(self):
        return self.out_dev.numel()


def scan_layers(sess: HybridSession, inputs: SuffixInputs, chunk, out_dtype=esc.DTYPE_F32, cold=False):
    """esc_scan_args for every linear layer: in-place state update on the session's fold states
    (cold=True: state_in = NULL, i.e. S_0 = 0)."""
    key = esc.shape_key_make(B, H, DK, DV, esc.DTYPE_BF16, out_dtype, chunk)
    if not key:
        raise ValueError("unsupported scan shape")
    T = inputs.T
    return [esc.scan_args(key, *inputs.dev[n], None if cold else sess.states[n], sess.states[n], inputs.out[n],
                          T, T, chunk) for n in range(len(sess.lin))], key
