"""B200-native hot path of THOR (arXiv 2507.11603): Lyα Monte Carlo resonant-scattering random walk.

`paper_2507_11603_b200.thor` is the thin ctypes binding over the C-ABI in include/thor.h (libthor_b200.so, CUDA,
sm_100a only).  `paper_2507_11603_b200.workloads` builds the seeded synthetic inputs.  There is no CPU fallback:
every call into `thor` raises if the CUDA library is missing.
"""
__all__ = ["thor", "workloads"]
