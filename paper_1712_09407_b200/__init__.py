"""B200-native TPC sector tracker (arXiv 1712.09407): CUDA kernels behind the C ABI of include/tpcst.h."""
from .binding import (EXPORTS, GLOBAL_DTYPE, MERGE_DTYPE, TPCST_DBG_BIN_OF, TPCST_DBG_BIN_START, TPCST_DBG_COUNTERS, TPCST_DBG_KERNEL_MS,
                      TPCST_DBG_LINKS, TPCST_DBG_LINKS_RAW, TPCST_DBG_OWNERS, TPCST_DBG_ROW_HITS, TPCST_DBG_STARTS,
                      TPCST_DBG_TRACKLETS, TPCST_DBG_WORK, TPCST_DEVICE, TPCST_ERR_ARG, TPCST_ERR_CAPACITY, TPCST_ERR_CUDA,
                      TPCST_ERR_RANGE, TPCST_ERR_STATE, TPCST_ERR_STATIC_LIMIT, TPCST_STATIC_MAX_CLUSTERS, TPCST_HOST_PAGEABLE, TPCST_HOST_PINNED, TPCST_N_SLOTS,
                      TPCST_OK, TRACK_DTYPE, WORK_NAMES, SectorTracker, TpcstError, TrackResult, lib, select_owners_static, selftest_random_access, selftest_math, tpcst_cuts,
                      tpcst_default_cuts, tpcst_geometry, tpcst_workspace_bytes)
from .build import build

__all__ = [n for n in dir() if not n.startswith("_")]
