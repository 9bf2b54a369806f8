"""B200-native Image Domain Gridding hot path (arXiv 1909.07226).

``synth`` (input generators) is importable on its own; the C-ABI binding is loaded
lazily by ``paper_1909_07226_b200.binding`` and fails loudly if the CUDA library is
missing -- there is no CPU fallback.
"""
__all__ = ["synth", "binding"]
