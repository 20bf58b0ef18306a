"""B200-native DF J/K build with INT8-emulated FP64 GEMMs (arXiv 2601.08077).

The product is the C-ABI library `libdfemul.so` (include/df_emul.h); this package is
its thin ctypes binding (`binding`, loaded on first attribute access so that
`python -m paper_2601_08077_b200.build` can run before the library exists).  There is
no CPU fallback: touching any entry point raises ImportError if the library has not
been built, and DFError(DF_ERR_DEVICE) on a machine without an sm_100 GPU.
"""
import importlib

_EXPORTS = (
    "DFError", "Workspace", "Context", "Plan", "EXPORTS", "lib", "lib_path",
    "DF_MODE_NOMINAL", "DF_MODE_GUARDED", "DF_STATUS_NONFINITE", "DF_STATUS_RANGE",
    "df_slices_for_tol", "df_num_int8_gemms", "df_kflush", "df_set_policy_mode", "df_plane_pitch",
    "df_emul_gemm_workspace_bytes", "df_jk_workspace_bytes", "df_jk_workspace_bytes_blocks", "df_set_workspace",
    "df_emul_gemm", "df_emul_gemm_slices", "df_jk_build", "df_jk_build_slices", "df_last_status", "df_screen_stats",
    "df_jk_plan_bytes", "df_jk_planned_workspace_bytes", "df_jk_build_planned", "df_jk_build_planned_slices",
    "df_debug_split_rows", "df_debug_split_cols", "df_debug_weight_sums", "df_debug_jk_build",
    "df_debug_set_gemm_flags", "df_launch_count", "df_profile_enable", "df_profile_read", "df_debug_mma_peak",
)
__all__ = list(_EXPORTS)


def __getattr__(name):
    if name in _EXPORTS:
        return getattr(importlib.import_module(".binding", __name__), name)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")
