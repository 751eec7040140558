"""B200-native (sm_100a) energy-and-force hot path of arxiv 2509.21694 behind a C ABI.

`binding` is a thin ctypes layer over `libmlip_b200.so` (include/mlip.h): argument marshalling
only, every step runs in the library's CUDA kernels. Importing this package does not load the
library; the first call does, and fails loudly if it is missing or no B200 is present.
"""
from .binding import (MLIP_BF16, MLIP_FP32, MLIP_MD_LANGEVIN, MLIP_MD_NVE, MLIP_SCAN_NOALLOC_MAX, Context, Graph, MlipError, Model, Partition,  # noqa: F401
                      energy_forces, energy_forces_shard, energy_forces_stress, lib_path, load_library, md_nve, md_run,
                      scan_i32, scan_i32_noalloc, step_host)
