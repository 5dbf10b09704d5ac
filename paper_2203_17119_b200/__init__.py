"""B200-native domain-wall-fermion hot path (arXiv:2203.17119).

The package is import-light on purpose: importing it does NOT load the CUDA
library, so `paper_2203_17119_b200.inputs` (the seeded input generators shared
by the tests' oracle side and the CUDA side) can be used on a CPU-only box.
The CUDA path lives in `paper_2203_17119_b200.api` and fails loudly when the
compiled C-ABI library is missing.
"""

__all__ = ["inputs", "api", "build"]
