"""paper_2005_09316_b200 -- B200-native WODEN visibility-prediction hot path.

`inputs` (seeded synthetic workloads) imports nothing heavy; `binding` loads the CUDA C-ABI
library (libwoden_b200.so) lazily and fails loudly when it is missing -- there is no CPU
fallback anywhere in this package.
"""
__all__ = ["inputs", "binding", "build", "parallel"]
