"""B200-native (sm_100a, fp64) hot path of the second-order dynamical low-rank integrator for the 6D
Vlasov-Poisson equations (arXiv 2110.13481, Algorithm 2).  `inputs` holds the seeded workload generators;
`dlr` is the thin ctypes binding of the C ABI in include/dlr.h (loaded lazily: importing this package
does not need the CUDA library, using `dlr` does and fails loudly without it)."""
__all__ = ["inputs", "dlr"]
