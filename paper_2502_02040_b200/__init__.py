"""paper_2502_02040_b200 — B200-native (sm_100a) implementation of the M2R2 decode hot path.

Public surface = the C ABI of include/m2r2.h (libm2r2.so) plus this thin binding.
"""
from .binding import (Engine, M2R2Error, Profile, PROF_CLASSES, lib, make_config, EXPORTS, Config, Sizes, Stats,  # noqa: F401
                      OK, INVALID_ARG, BAD_STATE, CAPACITY, CUDA, UNSUPPORTED, FP32, BF16,
                      POLICY_FIXED, POLICY_LRU, POLICY_LRU_AOT, POLICY_LRU_RANDOM, POLICY_LRU_PREV,
                      DBG_H, DBG_P, DBG_LOGITS, DBG_EXIT_LOGITS, DBG_K, DBG_V,
                      DBG_ROUTE_IDX, DBG_ROUTE_W, DBG_PRED_IDX, DBG_EXIT_SCORE,
                      final_head_noalloc, NOALLOC_MAX_ROWS, NOALLOC_MAX_D)
