"""B200-native DF J/K build with INT8-emulated FP64 GEMMs (arXiv 2601.08077).

The product is the C-ABI library `libdfemul.so` (include/df_emul.h); this package is
its thin ctypes binding.  There is no CPU fallback: importing `binding` raises if the
library has not been built (python -m paper_2601_08077_b200.build).
"""
from .binding import (  # noqa: F401
    DFError,
    Workspace,
    df_debug_jk_build,
    df_debug_mma_peak,
    df_debug_split_cols,
    df_debug_split_rows,
    df_debug_weight_sums,
    df_emul_gemm,
    df_emul_gemm_slices,
    df_emul_gemm_workspace_bytes,
    df_jk_build,
    df_jk_build_slices,
    df_jk_workspace_bytes,
    df_kflush,
    df_last_status,
    df_launch_count,
    df_num_int8_gemms,
    df_plane_pitch,
    df_set_policy_mode,
    df_set_workspace,
    df_slices_for_tol,
    lib,
    lib_path,
)
