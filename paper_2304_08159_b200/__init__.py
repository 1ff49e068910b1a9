"""B200-native pressure projection (after WaterLily.jl, arXiv 2304.08159): divergence, Geometric-MultiGrid solve of the
BDIM-modified Poisson system, pressure-gradient correction — hand-written CUDA for sm_100a behind the C ABI of
include/wl.h.

    from paper_2304_08159_b200 import binding as wl     # ctypes binding, same names as the C entry points
    from paper_2304_08159_b200 import synth             # seeded synthetic inputs (L, u)

Importing the package loads nothing; the first ``binding`` call loads libwl.so and raises if it is missing
(no CPU fallback exists).
"""
__all__ = ["binding", "synth", "build"]
