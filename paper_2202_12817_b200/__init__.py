"""B200-native incoherent harmonic sum (arXiv 2202.12817): greedy and PRESTO-like forms.

The product is the C-ABI library declared in ``include/hs.h`` (hand-written sm_100a kernels in
``csrc/``); ``binding`` is a thin ctypes marshalling layer with the same names; ``inputs`` holds
the seeded synthetic workloads (no method arithmetic).  There is no CPU fallback: every
``hs_*`` call fails loudly if the CUDA library is missing.
"""
__all__ = ["inputs", "binding"]
