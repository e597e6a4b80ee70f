"""paper_1107_5463_b200 -- B200-native checkerboard Metropolis sweeps for O(n) lattice spin models
(Weigel & Yavors'kii, arXiv:1107.5463): libspin.so (CUDA, C ABI in include/spin.h) and its thin binding."""
from . import workloads  # noqa: F401
from .binding import (  # noqa: F401
    INIT_COLD, INIT_HOT, OPT_PLAIN_KERNELS, OPT_TMA_KERNELS, OPT_L2_PREFETCH, OPT_KERNEL_VARIANT, OPT_TEMPORAL_BLOCKING, OPT_TBLOCK_ROWS, OPT_L2_KEEP, OPT_DEFER_CAP, UPDATE_HEATBATH, UPDATE_METROPOLIS, SpinError, SpinSystem, from_workload, lib, lib_path, make_config, workspace_bytes,
)
