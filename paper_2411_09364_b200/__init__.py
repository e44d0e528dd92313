"""B200-native (sm_100a, fp64 CUDA) hot path of CaLES (arXiv 2411.09364): one low-storage RK3 step of the
incompressible staggered-grid LES behind the C ABI of include/cales.h.

`from paper_2411_09364_b200 import binding` loads libcales.so (and fails loudly if it is not built);
`inputs` holds the seeded synthetic workloads and imports nothing else from the package.
"""
__all__ = ["binding", "inputs", "build"]
