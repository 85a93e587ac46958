"""B200-native coupled ACM lattice-Boltzmann step (arXiv 2012.06144) behind a C ABI.

`binding` holds the thin ctypes layer over libacm.so (same names as include/acm.h);
`inputs` holds the seeded synthetic workloads; `build` compiles the library in-tree.
Importing the package does not load CUDA; using `binding` without a built libacm.so or
without a CUDA device fails loudly -- there is no CPU fallback.
"""
__all__ = ["binding", "inputs", "build"]
