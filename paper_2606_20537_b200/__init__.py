"""esc — execution-state capsules on B200 (sm_100a).

B200-native hot path of arxiv/paper_2606_20537: capsule snapshot / restore / fork / rollback
(single-launch descriptor-table copy kernel) and the chunked gated linear-attention scan,
behind the C-ABI declared in include/esc.h.  `esc` (the ctypes binding over libesc.so) is
imported lazily so that `synth` (seeded inputs, no method arithmetic) stays importable on a
box without the CUDA library; every call into the path fails loudly if libesc.so is missing.
"""
__all__ = ["esc", "synth"]


def __getattr__(name):
    if name in ("esc", "synth"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
