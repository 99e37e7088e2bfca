"""B200-native hydro hot path (arxiv 2007.05218): Python binding of the C-ABI library.

`workloads` (input generation only) is importable without a GPU.  Everything that
computes lives in csrc/ behind include/hydro.h and is reached through `binding`, which
raises at call time if libhydro_b200.so is missing -- there is no CPU fallback.
"""
__all__ = ["workloads", "binding"]
