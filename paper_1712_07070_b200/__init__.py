"""B200-native batched patch-group hydrodynamic solver (the hot path of GAMER-2, arXiv 1712.07070).

`paper_1712_07070_b200.binding` is the thin ctypes layer over the C-ABI library
(include/gamer_hydro.h); `paper_1712_07070_b200.inputs` builds the seeded synthetic workloads.
The CUDA library is loaded lazily by the binding and fails loudly if it is missing: there is
no CPU fallback anywhere in this package.
"""
__all__ = ["binding", "inputs"]
