"""B200-native coupled T-matrix multiple-scattering solver (hot path of arXiv 2107.09879).

`workloads` (numpy only) generates the seeded synthetic inputs; `libtm` is the thin ctypes binding
over the C-ABI CUDA library (include/tm.h).  The CUDA library is loaded on first use of `libtm`
and its absence is a hard error: there is no CPU fallback.
"""
__all__ = ["workloads", "libtm"]
