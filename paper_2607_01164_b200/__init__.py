"""B200-native W-VEG sampler (hot path of arxiv/paper_2607_01164): C-ABI CUDA library + thin binding.

``inputs`` holds the seeded synthetic workloads (no method arithmetic); ``api`` is the ctypes
binding of include/gs.h; ``build`` compiles ``libgs.so`` for sm_100a.  Nothing here imports the
oracle, and there is no CPU fallback.
"""
__all__ = ["api", "inputs", "build"]
