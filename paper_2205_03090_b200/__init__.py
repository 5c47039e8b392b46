"""paper_2205_03090_b200 -- B200-native batched isothermal two-phase SRK flash (PTFlash hot path).

The product is libptflash.so (C ABI in include/ptflash.h, CUDA kernels in csrc/).  `binding` marshals
arguments; `workloads` holds the seeded synthetic inputs; `build` compiles the library in-tree.
Nothing here imports the CPU oracle (oracle/), which is test infrastructure.
"""
from . import workloads  # noqa: F401  (numpy only; importable without the CUDA library)

__all__ = ["workloads", "binding", "build"]
