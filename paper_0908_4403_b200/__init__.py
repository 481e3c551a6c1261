"""B200-native (sm_100a) hot path of arXiv 0908.4403 (HEGET): summed squared helicity
amplitudes of u ubar -> n gamma behind the C ABI of include/heget.h."""
from . import workloads  # noqa: F401
from .binding import (ALGO_SUBSET, ALGO_TREE, ALGO_TREE2, FP32, FP64, GEN_FIXED, GEN_LOGUNIFORM, GEN_TOYPDF,  # noqa: F401
                      OBS_DR_ALL, OBS_DR_MIN, OBS_PT_MAX, Heget, HegetError, load_library)
