"""paper_1609_00724_b200: B200-native (sm_100a CUDA) field-line tracer / squashing factor Q / FLEDGE / refinement,
after Tassev & Savcheva, "QSL Squasher" (arXiv:1609.00724).  The product is the C-ABI library libqsl.so
(include/qsl.h); this package is its thin Python binding."""
from .binding import (  # noqa: F401
    QSL_F32, QSL_F64, QSL_NORMALIZE_FIRST, QSL_INTERP_FIRST, QSL_RK4, QSL_EULER, QSL_CK45, QSL_TRACE_L, QSL_TRACE_LQ,
    QSL_ARITH_F64, QSL_ARITH_F32, QSL_TRILINEAR, QSL_TRIQUADRATIC, QSL_TRICUBIC, QSL_CARTESIAN, QSL_SPHERICAL, QSL_LAYOUT_CELL_TABLE, QSL_LAYOUT_NODES_ONLY, QSL_LAYOUT_CELL_TABLE_F32, QSL_LAYOUT_CELL_TABLES_BOTH, QSL_ST_SEED_OUTSIDE, QSL_ST_NULL_AT_SEED, QSL_ST_STALL_F, QSL_ST_STALL_B,
    QSL_ST_CAP_F, QSL_ST_CAP_B, QSL_ST_OPEN, QSL_FLAG_NO_SORT, QSL_FLAG_NO_REFILL, QSL_FLAG_KERNEL_V1, QSL_FLAG_KERNEL_FRAME,
    QslError, Field, lib, LIB_PATH, peaks_lib, PEAKS_LIB_PATH, make_lattice, make_trace_params, qsl_field_create, qsl_trace, qsl_fledge_dense,
    qsl_fledge_sparse, qsl_select, qsl_refine, qsl_refine_noalloc, QSL_REFINE_NOALLOC_MAX_CELLS, DEFAULT_OUTPUTS, qsl_profile_enable, qsl_profile_trace_kernel_ms, qsl_peak_fma,
    qsl_peak_gather, qsl_hilbert_bits, qsl_hilbert_level0, qsl_hilbert_keys, qsl_hilbert_cells, qsl_sort_keys64, qsl_gather,
    qsl_hilbert_refine, qsl_hilbert_merge, qsl_hilbert_convert,
)
from .driver import adaptive_map, hilbert_map, trace_host  # noqa: F401,E402
