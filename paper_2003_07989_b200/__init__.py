"""B200-native hot path of Vietoris-Rips barcode computation (arXiv 2003.07989): filtration
construction with clearing and apparent-pair finding, hand-written CUDA for sm_100a behind the C ABI
of include/rips.h.  `rips` is the thin ctypes binding, `inputs` the seeded synthetic workloads,
`build` compiles the shared library in-tree."""
__all__ = ["rips", "inputs", "build"]
