"""libprepos: the data-parallel hot path of speculative pre-positioning (arxiv/paper_2606_29565) on B200.

`paper_2606_29565_b200.prepos` is the thin ctypes binding over the C-ABI library declared in
include/prepos.h; `paper_2606_29565_b200.synth` holds the seeded input generators.  Nothing is
imported eagerly so the generators stay usable where the CUDA library is absent; every op of
`prepos` raises if libprepos.so cannot be loaded -- there is no CPU fallback.
"""
__all__ = ["prepos", "synth"]
