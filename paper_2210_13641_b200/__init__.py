"""nsm — B200-native NeRF-SLAM mapping step (arxiv 2210.13641): Python binding of libnsm.so.

The product is the C-ABI library declared in include/nsm.h (hand-written CUDA for sm_100a);
this package only marshals arguments.  Importing it never falls back to a CPU path.
"""
from .binding import (DEBUG_ITEMS, EXPORTS, LIB_PATH, NSM_MLP_BF16, NSM_MLP_FP16, NSM_MLP_FP32,
                      NSM_OCC_FROM_FIELD, NSM_OCC_FULL, NSM_OCC_SET, NSM_OPT_BATCH_READY, NSM_OPT_DEBUG_TIMELINE, NSM_OPT_POSE_GRADIENTS, NSM_OPT_POSE_LEVELS, DeviceBatch, Field, HostBatch,
                      MarchBuffers, NsmError, NSM_MARCH_STATIC_MAX_RAYS, load_library, make_config, nsm_march_static)

__all__ = ["Field", "DeviceBatch", "HostBatch", "NsmError", "load_library", "make_config", "EXPORTS",
           "LIB_PATH", "DEBUG_ITEMS", "NSM_MLP_FP32", "NSM_MLP_FP16", "NSM_MLP_BF16", "NSM_OCC_FULL", "NSM_OPT_BATCH_READY", "NSM_OPT_POSE_GRADIENTS",
           "NSM_OCC_SET", "NSM_OCC_FROM_FIELD", "NSM_OPT_DEBUG_TIMELINE", "NSM_OPT_POSE_LEVELS",
           "MarchBuffers", "nsm_march_static", "NSM_MARCH_STATIC_MAX_RAYS"]
