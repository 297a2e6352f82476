"""libmopal - B200-native FP64 n-body kick / encounter flagging / Kepler drift
(the data-parallel hot path of Mercury-Opal, arxiv 2601.19654).

``workloads`` (seeded inputs, numpy only) imports nothing else.  The CUDA
binding lives in ``paper_2601_19654_b200.mopal`` and is imported lazily so that
the input generators stay usable without the compiled library; every compute
entry point fails loudly when ``libmopal.so`` or a CUDA device is missing -
there is no CPU fallback.
"""
__all__ = ["workloads", "mopal"]
