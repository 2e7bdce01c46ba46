"""paper_2505_14372_b200 — B200-native hot path of mixed-state multislice ptychography (arxiv 2505.14372).

`ptycho` is the thin binding over the C-ABI library (include/ptycho.h); `synth` builds seeded inputs.
The binding loads the CUDA library lazily and fails loudly if it is missing: there is no CPU fallback.
"""
__all__ = ["ptycho", "synth"]
