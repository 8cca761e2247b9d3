"""B200-native parallel-rejection kinetic Monte Carlo for Coulomb glasses (arXiv 1407.5026).

The product is libcg.so (C ABI in include/cg.h, CUDA in csrc/cg.cu); this package is its thin
ctypes binding.  See DESIGN.md.
"""
from .binding import CgError, CoulombGlass, bench_l2, run_many, lib, EXPORTS  # noqa: F401
