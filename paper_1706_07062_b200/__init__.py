"""B200-native batched Kerr-Schild geodesic integrator (hot path of GRay2, arXiv:1706.07062).

``paper_1706_07062_b200.gray2`` is the thin ctypes binding over the C-ABI library
(include/gray2.h); ``paper_1706_07062_b200.inputs`` holds the seeded synthetic input recipes.
Nothing here imports the CPU oracle, and there is no CPU fallback.
"""
__all__ = ["gray2", "inputs"]
