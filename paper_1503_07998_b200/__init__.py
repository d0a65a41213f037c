"""B200-native plane-wise multi-view Richardson-Lucy deconvolution (arXiv 1503.07998).

`synth` (seeded inputs) imports without a GPU.  The compute API lives in `binding` and is loaded
lazily: it needs the in-tree CUDA library (`libmvd.so`, built by `build.py`) and FAILS LOUDLY if
that library is missing -- there is no CPU fallback.
"""
__all__ = ["synth", "binding", "build"]
