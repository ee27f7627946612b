"""B200-native CSC narrow-band signed distance transform (arXiv:1903.00353 hot path).

`paper_1903_00353_b200.workloads` : seeded synthetic inputs (no method arithmetic).
`paper_1903_00353_b200.binding`   : thin ctypes binding over the C-ABI library
                                     (`include/sdf.h`); loaded lazily, fails loudly if the
                                     CUDA library is missing.
"""
__all__ = ["workloads", "binding"]
