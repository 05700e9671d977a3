"""fizzy-b200: B200-native (sm_100a, fp64) RK3 substep of the CaNS-Fizzy two-phase solver
(arXiv 2502.04189).  The product is the C-ABI library `libfizzy.so` (include/fizzy.h); this
package holds its CUDA sources (csrc/), the build step (build.py), a thin ctypes binding with
the same entry-point names (binding.py) and the seeded workload generators (workloads.py).

Importing the package does not load the CUDA library; `paper_2502_04189_b200.binding` does,
and fails loudly when it is missing."""

__all__ = ["workloads"]
