"""libctr: B200-native (sm_100a) hot path of edge-preserving-TV CT reconstruction
(arxiv/paper_1009_2288). The product is the C-ABI library `libctr.so` (include/ctr.h,
csrc/*.cu); this package is its thin Python binding. There is no CPU fallback.
"""
from .binding import (CtrError, Handle, ctr_create, ctr_destroy, ctr_geometry, ctr_params,
                      ctr_sweep_stat, load_library, make_geometry, make_params, EXPORTS, CTR_GEOM_NO_TABLES, CTR_GEOM_NO_GRAPHS, CTR_GEOM_NO_STORED_P, CTR_GEOM_NO_LAZY_CGLS,
                      ctr_peaks, ctr_measure_peaks, ctr_forward_noalloc)

__all__ = ["CtrError", "Handle", "ctr_create", "ctr_destroy", "ctr_geometry", "ctr_params",
           "ctr_sweep_stat", "load_library", "make_geometry", "make_params", "EXPORTS", "CTR_GEOM_NO_TABLES", "CTR_GEOM_NO_GRAPHS", "CTR_GEOM_NO_STORED_P", "ctr_peaks", "ctr_measure_peaks", "ctr_forward_noalloc"]
