"""B200-native Linac hot path: RREF / null space over F_p and an fp64 solve (hand-written CUDA).

The product is the C-ABI library `liblinac.so` (include/linac.h); this package is its thin
Python binding.  Build with `python -m paper_2605_25863_b200.build`.
"""
from . import linac  # noqa: F401
from .linac import (  # noqa: F401
    LinacError, rref_u32, rref_u64, nullspace_u32, nullspace_from_rref_u32, solve_u32, rank_factor_u32, load_matrix_u32, solve_f64, rref_f64, rref_c128, gemm_sub_u32, gemm_sub_u32_static, set_option, last_stats, last_marks,
    release_workspace, version, measure_peak,
)
