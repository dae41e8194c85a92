"""heget-b200: B200-native evaluation of helicity- and colour-summed tree-level QCD matrix elements (arXiv:0909.5257)."""
from .heget import (Process, HegetError, Cuts, Info, lib, launch_count, shard_range, fma_probe, LIB_PATH, EXPORTS,
                    FP64, FP32, FP32X2, HEL_SUM, HEL_SAMPLE, HEL_FIXED, OK, EINVAL, EUNSUPPORTED, ECUDA, ENOMEM, ECOMPILE,
                    KERNEL_AUTO, KERNEL_STRAIGHT, KERNEL_TABLE)
