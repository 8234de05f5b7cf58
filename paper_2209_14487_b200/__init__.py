"""B200-native crowd move of arXiv:2209.14487: thin binding over the C-ABI library libqmc_crowd.so.

The product is the CUDA library (csrc/, include/qmc_crowd.h); this package only marshals arguments.
"""
from .binding import (Crowd, CrowdDesc, QmcError, EXPORTS, QMC_OPT_GRAPH, QMC_OPT_PROFILE, QMC_OPT_SUBCROWDS, QMC_OPT_RECOMPUTE_EVERY, QMC_OPT_STRIP_ROWS, KERNEL_CLASSES, QMC_OK, QMC_ERR_INVALID_ARG,  # noqa: F401
                      QMC_ERR_CUDA, QMC_ERR_WORKSPACE, QMC_ERR_SINGULAR, QMC_ERR_STATE, lib_path, load, qmc_spo_vgl_static, STATIC_SCRATCH_BYTES)
