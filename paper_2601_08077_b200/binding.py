"""ctypes binding of libdfemul.so -- argument marshalling only (include/df_emul.h).

Every function here has the name and argument order of the C entry point it calls;
tensors are passed as `data_ptr()` and the stream as
`torch.cuda.current_stream().cuda_stream`.  PyTorch is used for device memory and
streams only.  Nothing is computed in Python and nothing falls back to the CPU: a
missing library raises ImportError, a failing call raises DFError.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
lib_path = os.path.join(_HERE, "libdfemul.so")

if not os.path.exists(lib_path):
    raise ImportError(
        f"{lib_path} is missing: build it with `python -m paper_2601_08077_b200.build` "
        "(there is no CPU fallback)"
    )
lib = C.CDLL(lib_path)

DF_MODE_NOMINAL, DF_MODE_GUARDED = 0, 1
DF_STATUS_NONFINITE, DF_STATUS_RANGE = 1, 2
_ERRORS = {
    -1: "DF_ERR_NULL", -2: "DF_ERR_DIM", -3: "DF_ERR_TOL", -4: "DF_ERR_WORKSPACE",
    -5: "DF_ERR_DEVICE", -6: "DF_ERR_CUDA", -7: "DF_ERR_ALIGN", -8: "DF_ERR_TOO_LARGE",
}


class DFError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what} failed: {_ERRORS.get(code, code)}")
        self.code = code


_vp, _i64, _i32, _f64 = C.c_void_p, C.c_int64, C.c_int, C.c_double
_SIG = {
    "df_slices_for_tol": (_i32, [_f64, _i32]),
    "df_num_int8_gemms": (_i32, [_i32]),
    "df_kflush": (_i32, [_i32]),
    "df_set_policy_mode": (_i32, [_i32]),
    "df_plane_pitch": (_i64, [_i64]),
    "df_emul_gemm_workspace_bytes": (_i64, [_i64, _i64, _i64, _i32]),
    "df_jk_workspace_bytes": (_i64, [_i64, _i64, _i64, _i32]),
    "df_jk_workspace_bytes_blocks": (_i64, [_i64, _i64, _i64, _i32, _i64]),
    "df_set_workspace": (_i32, [_vp, _i64]),
    "df_emul_gemm": (_i32, [_vp, _vp, _vp, _i64, _i64, _i64, _f64, _vp]),
    "df_emul_gemm_slices": (_i32, [_vp, _vp, _vp, _i64, _i64, _i64, _i32, _vp]),
    "df_emul_gemm_static": (_i32, [_vp, _vp, _vp, _i64, _i64, _i64, _f64, _vp]),
    "df_emul_gemm_static_scratch_bytes": (_i64, []),
    "df_jk_build": (_i32, [_vp, _i64, _i64, _vp, _i64, _vp, _f64, _vp, _vp, _vp]),
    "df_jk_build_slices": (_i32, [_vp, _i64, _i64, _vp, _i64, _vp, _i32, _vp, _vp, _vp]),
    "df_jk_plan_bytes": (_i64, [_i64, _i64, _i32]),
    "df_jk_plan_create": (_i32, [_vp, _i64, _i64, _i32, _vp, _i64, _vp]),
    "df_jk_planned_workspace_bytes": (_i64, [_i64, _i64, _i64, _i32, _i64]),
    "df_jk_build_planned": (_i32, [_vp, _i32, _vp, _i64, _i64, _vp, _i64, _vp, _f64, _vp, _vp, _vp]),
    "df_jk_build_planned_slices": (_i32, [_vp, _i32, _vp, _i64, _i64, _vp, _i64, _vp, _i32, _vp, _vp, _vp]),
    "df_last_status": (_i32, [_vp, C.POINTER(C.c_int)]),
    "df_context_create": (_i32, [_vp, _i64, C.POINTER(_vp)]),
    "df_context_destroy": (_i32, [_vp]),
    "df_context_set_policy_mode": (_i32, [_vp, _i32]),
    "df_context_set_debug_flags": (_i32, [_vp, _i32]),
    "df_context_emul_gemm": (_i32, [_vp, _vp, _vp, _vp, _i64, _i64, _i64, _f64, _vp]),
    "df_context_emul_gemm_slices": (_i32, [_vp, _vp, _vp, _vp, _i64, _i64, _i64, _i32, _vp]),
    "df_context_jk_build": (_i32, [_vp, _vp, _i64, _i64, _vp, _i64, _vp, _f64, _vp, _vp, _vp]),
    "df_context_jk_build_slices": (_i32, [_vp, _vp, _i64, _i64, _vp, _i64, _vp, _i32, _vp, _vp, _vp]),
    "df_context_jk_plan_create": (_i32, [_vp, _vp, _i64, _i64, _i32, _vp, _i64, _vp]),
    "df_context_jk_build_planned": (_i32, [_vp, _vp, _i32, _vp, _i64, _i64, _vp, _i64, _vp, _f64, _vp, _vp, _vp]),
    "df_context_jk_build_planned_slices": (_i32, [_vp, _vp, _i32, _vp, _i64, _i64, _vp, _i64, _vp, _i32, _vp, _vp, _vp]),
    "df_context_last_status": (_i32, [_vp, _vp, C.POINTER(C.c_int)]),
    "df_context_screen_stats": (_i32, [_vp, _vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]),
    "df_screen_stats": (_i32, [_vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]),
    "df_debug_split_rows": (_i32, [_vp, _i64, _i64, _i32, _vp, _vp, _vp]),
    "df_debug_split_cols": (_i32, [_vp, _i64, _i64, _i32, _vp, _vp, _vp]),
    "df_debug_weight_sums": (_i32, [_vp, _vp, _i64, _i64, _i64, _i32, _i32, _i32, _vp, _vp]),
    "df_debug_jk_build": (_i32, [_vp, _i64, _i64, _vp, _i64, _vp, _i32, _vp, _vp, _vp, _vp,
                                 C.POINTER(C.c_int), _vp]),
    "df_debug_set_gemm_flags": (_i32, [_i32]),
    "df_launch_count": (_i64, []),
    "df_profile_enable": (_i32, [_i32]),
    "df_profile_num_classes": (_i32, []),
    "df_profile_class_name": (C.c_char_p, [_i32]),
    "df_profile_read": (_i32, [C.POINTER(C.c_float), C.POINTER(C.c_int)]),
    "df_debug_mma_peak": (_i32, [_i32, _i32, _i32, C.POINTER(C.c_float), _vp]),
}
EXPORTS = tuple(_SIG)
for _name, (_res, _args) in _SIG.items():
    _fn = getattr(lib, _name)  # AttributeError if the library does not export it
    _fn.restype, _fn.argtypes = _res, _args


def _check(code: int, what: str) -> int:
    if code < 0:
        raise DFError(int(code), what)
    return int(code)


def _stream(stream=None):
    if stream is not None:
        return C.c_void_p(int(stream))
    import torch

    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t, dtype=None):
    if t is None:
        return C.c_void_p(0)
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"expected dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


# ---- policy -------------------------------------------------------------------------------
def df_slices_for_tol(tol: float, mode: int = DF_MODE_GUARDED) -> int:
    return _check(lib.df_slices_for_tol(float(tol), int(mode)), "df_slices_for_tol")


def df_num_int8_gemms(s: int) -> int:
    return _check(lib.df_num_int8_gemms(int(s)), "df_num_int8_gemms")


def df_kflush(s: int) -> int:
    return _check(lib.df_kflush(int(s)), "df_kflush")


def df_set_policy_mode(mode: int) -> None:
    _check(lib.df_set_policy_mode(int(mode)), "df_set_policy_mode")


def df_plane_pitch(cols: int) -> int:
    return _check(lib.df_plane_pitch(int(cols)), "df_plane_pitch")


# ---- workspace ----------------------------------------------------------------------------
def df_emul_gemm_workspace_bytes(m: int, n: int, k: int, s: int) -> int:
    return _check(lib.df_emul_gemm_workspace_bytes(m, n, k, s), "df_emul_gemm_workspace_bytes")


def df_jk_workspace_bytes(nao: int, naux: int, nocc: int, s: int) -> int:
    return _check(lib.df_jk_workspace_bytes(nao, naux, nocc, s), "df_jk_workspace_bytes")


def df_jk_workspace_bytes_blocks(nao: int, naux: int, nocc: int, s: int, nblocks: int) -> int:
    return _check(lib.df_jk_workspace_bytes_blocks(nao, naux, nocc, s, nblocks), "df_jk_workspace_bytes_blocks")


def df_set_workspace(buf) -> None:
    """buf: a uint8 CUDA tensor (kept alive by the caller), or None to unregister."""
    if buf is None:
        _check(lib.df_set_workspace(None, 0), "df_set_workspace")
    else:
        _check(lib.df_set_workspace(_ptr(buf), buf.numel() * buf.element_size()), "df_set_workspace")


class Workspace:
    """Owns a device buffer and registers it as the library's workspace."""

    def __init__(self, nbytes: int, device="cuda"):
        import torch

        self.buf = torch.empty(int(nbytes) + 256, dtype=torch.uint8, device=device)
        off = (-self.buf.data_ptr()) % 256
        self.view = self.buf[off: off + int(nbytes)]
        df_set_workspace(self.view)

    def close(self):
        df_set_workspace(None)
        self.buf = self.view = None


class Context:
    """A df_context: owns a device buffer as its workspace.  One context per concurrent stream; the
    methods have the names and argument order of the df_context_* entry points (marshalling only)."""

    def __init__(self, nbytes: int, device="cuda"):
        import torch

        self.buf = torch.empty(int(nbytes) + 256, dtype=torch.uint8, device=device)
        off = (-self.buf.data_ptr()) % 256
        self.view = self.buf[off: off + int(nbytes)]
        h = _vp()
        with torch.cuda.device(self.buf.device):
            _check(lib.df_context_create(_ptr(self.view), int(nbytes), C.byref(h)), "df_context_create")
        self.handle = h

    def close(self):
        if self.handle is not None:
            _check(lib.df_context_destroy(self.handle), "df_context_destroy")
        self.handle = self.buf = self.view = None

    def set_policy_mode(self, mode: int) -> None:
        _check(lib.df_context_set_policy_mode(self.handle, int(mode)), "df_context_set_policy_mode")

    def set_debug_flags(self, flags: int) -> None:
        _check(lib.df_context_set_debug_flags(self.handle, int(flags)), "df_context_set_debug_flags")

    def emul_gemm(self, A, B, Cout, m, n, k, tol, stream=None) -> None:
        import torch

        f = torch.float64
        _check(lib.df_context_emul_gemm(self.handle, _ptr(A, f), _ptr(B, f), _ptr(Cout, f), m, n, k, float(tol),
                                        _stream(stream)), "df_context_emul_gemm")

    def emul_gemm_slices(self, A, B, Cout, m, n, k, s, stream=None) -> None:
        import torch

        f = torch.float64
        _check(lib.df_context_emul_gemm_slices(self.handle, _ptr(A, f), _ptr(B, f), _ptr(Cout, f), m, n, k, int(s),
                                               _stream(stream)), "df_context_emul_gemm_slices")

    def jk_build(self, B_packed, nao, naux, C_occ, nocc, D, tol, J, K, stream=None) -> None:
        import torch

        f = torch.float64
        _check(lib.df_context_jk_build(self.handle, _ptr(B_packed, f), nao, naux, _ptr(C_occ, f), nocc, _ptr(D, f),
                                       float(tol), _ptr(J, f), _ptr(K, f), _stream(stream)), "df_context_jk_build")

    def jk_build_slices(self, B_packed, nao, naux, C_occ, nocc, D, s, J, K, stream=None) -> None:
        import torch

        f = torch.float64
        _check(lib.df_context_jk_build_slices(self.handle, _ptr(B_packed, f), nao, naux, _ptr(C_occ, f), nocc,
                                              _ptr(D, f), int(s), _ptr(J, f), _ptr(K, f), _stream(stream)),
               "df_context_jk_build_slices")

    def jk_plan_create(self, B_packed, nao, naux, smax, plan_view, stream=None) -> None:
        import torch

        _check(lib.df_context_jk_plan_create(self.handle, _ptr(B_packed, torch.float64), nao, naux, int(smax),
                                             _ptr(plan_view), plan_view.numel(), _stream(stream)),
               "df_context_jk_plan_create")

    def jk_build_planned(self, plan, B_packed, nao, naux, C_occ, nocc, D, tol, J, K, stream=None) -> None:
        import torch

        f = torch.float64
        _check(lib.df_context_jk_build_planned(self.handle, _ptr(plan.view), plan.smax, _ptr(B_packed, f), nao, naux,
                                               _ptr(C_occ, f), nocc, _ptr(D, f), float(tol), _ptr(J, f), _ptr(K, f),
                                               _stream(stream)), "df_context_jk_build_planned")

    def jk_build_planned_slices(self, plan, B_packed, nao, naux, C_occ, nocc, D, s, J, K, stream=None) -> None:
        import torch

        f = torch.float64
        _check(lib.df_context_jk_build_planned_slices(self.handle, _ptr(plan.view), plan.smax, _ptr(B_packed, f), nao,
                                                      naux, _ptr(C_occ, f), nocc, _ptr(D, f), int(s), _ptr(J, f),
                                                      _ptr(K, f), _stream(stream)),
               "df_context_jk_build_planned_slices")

    def last_status(self, stream=None) -> int:
        out = C.c_int(0)
        _check(lib.df_context_last_status(self.handle, _stream(stream), C.byref(out)), "df_context_last_status")
        return int(out.value)

    def screen_stats(self, stream=None):
        a, t = C.c_int64(0), C.c_int64(0)
        _check(lib.df_context_screen_stats(self.handle, _stream(stream), C.byref(a), C.byref(t)),
               "df_context_screen_stats")
        return int(a.value), int(t.value)


# ---- the two entry points -----------------------------------------------------------------
def df_emul_gemm(A, B, Cout, m, n, k, tol, stream=None) -> None:
    import torch

    _check(lib.df_emul_gemm(_ptr(A, torch.float64), _ptr(B, torch.float64), _ptr(Cout, torch.float64),
                            m, n, k, float(tol), _stream(stream)), "df_emul_gemm")


def df_emul_gemm_slices(A, B, Cout, m, n, k, s, stream=None) -> None:
    import torch

    _check(lib.df_emul_gemm_slices(_ptr(A, torch.float64), _ptr(B, torch.float64), _ptr(Cout, torch.float64),
                                   m, n, k, int(s), _stream(stream)), "df_emul_gemm_slices")


def df_emul_gemm_static(A, B, Cout, m, n, k, tol, stream=None) -> None:
    """df_emul_gemm for callers that cannot allocate device memory: no workspace is registered or
    needed, the scratch is a 64 MiB array built into the library (include/df_emul.h).  Raises DFError
    with code -8 (DF_ERR_TOO_LARGE) when the sizes need more than that; calls that may overlap on the
    GPU must not share it."""
    import torch

    _check(lib.df_emul_gemm_static(_ptr(A, torch.float64), _ptr(B, torch.float64), _ptr(Cout, torch.float64),
                                   m, n, k, float(tol), _stream(stream)), "df_emul_gemm_static")


def df_emul_gemm_static_scratch_bytes() -> int:
    return int(lib.df_emul_gemm_static_scratch_bytes())


def df_jk_build(B_packed, nao, naux, C_occ, nocc, D, tol, J, K, stream=None) -> None:
    import torch

    f = torch.float64
    _check(lib.df_jk_build(_ptr(B_packed, f), nao, naux, _ptr(C_occ, f), nocc, _ptr(D, f), float(tol),
                           _ptr(J, f), _ptr(K, f), _stream(stream)), "df_jk_build")


def df_jk_build_slices(B_packed, nao, naux, C_occ, nocc, D, s, J, K, stream=None) -> None:
    import torch

    f = torch.float64
    _check(lib.df_jk_build_slices(_ptr(B_packed, f), nao, naux, _ptr(C_occ, f), nocc, _ptr(D, f), int(s),
                                  _ptr(J, f), _ptr(K, f), _stream(stream)), "df_jk_build_slices")


# ---- plan: B split once for a whole SCF ---------------------------------------------------
def df_jk_plan_bytes(nao: int, naux: int, smax: int) -> int:
    return _check(lib.df_jk_plan_bytes(nao, naux, int(smax)), "df_jk_plan_bytes")


def df_jk_planned_workspace_bytes(nao: int, naux: int, nocc: int, s: int, nblocks: int) -> int:
    return _check(lib.df_jk_planned_workspace_bytes(nao, naux, nocc, s, nblocks), "df_jk_planned_workspace_bytes")


class Plan:
    """Owns the device buffer of a plan and fills it from B_packed (a workspace must be registered)."""

    def __init__(self, B_packed, nao: int, naux: int, smax: int, stream=None):
        import torch

        self.nao, self.naux, self.smax = int(nao), int(naux), int(smax)
        nbytes = df_jk_plan_bytes(nao, naux, smax)
        self.buf = torch.empty(nbytes + 256, dtype=torch.uint8, device=B_packed.device)
        off = (-self.buf.data_ptr()) % 256
        self.view = self.buf[off: off + nbytes]
        _check(lib.df_jk_plan_create(_ptr(B_packed, torch.float64), nao, naux, int(smax), _ptr(self.view), nbytes,
                                     _stream(stream)), "df_jk_plan_create")

    def close(self):
        self.buf = self.view = None


def df_jk_build_planned(plan, B_packed, nao, naux, C_occ, nocc, D, tol, J, K, stream=None) -> None:
    import torch

    f = torch.float64
    _check(lib.df_jk_build_planned(_ptr(plan.view), plan.smax, _ptr(B_packed, f), nao, naux, _ptr(C_occ, f), nocc,
                                   _ptr(D, f), float(tol), _ptr(J, f), _ptr(K, f), _stream(stream)),
           "df_jk_build_planned")


def df_jk_build_planned_slices(plan, B_packed, nao, naux, C_occ, nocc, D, s, J, K, stream=None) -> None:
    import torch

    f = torch.float64
    _check(lib.df_jk_build_planned_slices(_ptr(plan.view), plan.smax, _ptr(B_packed, f), nao, naux, _ptr(C_occ, f),
                                          nocc, _ptr(D, f), int(s), _ptr(J, f), _ptr(K, f), _stream(stream)),
           "df_jk_build_planned_slices")


def df_last_status(stream=None) -> int:
    out = C.c_int(0)
    _check(lib.df_last_status(_stream(stream), C.byref(out)), "df_last_status")
    return int(out.value)


def df_screen_stats(stream=None):
    """(active, total) K blocks of GEMM(5)'s left operand since the last call; synchronises."""
    a, t = C.c_int64(0), C.c_int64(0)
    _check(lib.df_screen_stats(_stream(stream), C.byref(a), C.byref(t)), "df_screen_stats")
    return int(a.value), int(t.value)


# ---- debug exports ------------------------------------------------------------------------
def df_debug_split_rows(X, rows, cols, s, e, planes, stream=None) -> None:
    import torch

    _check(lib.df_debug_split_rows(_ptr(X, torch.float64), rows, cols, int(s), _ptr(e, torch.int32),
                                   _ptr(planes, torch.int8), _stream(stream)), "df_debug_split_rows")


def df_debug_split_cols(X, k, n, s, e, planes, stream=None) -> None:
    import torch

    _check(lib.df_debug_split_cols(_ptr(X, torch.float64), k, n, int(s), _ptr(e, torch.int32),
                                   _ptr(planes, torch.int8), _stream(stream)), "df_debug_split_cols")


def df_debug_weight_sums(DA, DB, m, n, k, s, chunk, bk, P, stream=None) -> None:
    import torch

    _check(lib.df_debug_weight_sums(_ptr(DA, torch.int8), _ptr(DB, torch.int8), m, n, k, int(s), int(chunk),
                                    int(bk), _ptr(P, torch.int32), _stream(stream)), "df_debug_weight_sums")


def df_debug_jk_build(B_packed, nao, naux, C_occ, nocc, D, s, J, K, X_out=None, e6_out=None, stream=None) -> int:
    import torch

    f = torch.float64
    ng = C.c_int(0)
    _check(lib.df_debug_jk_build(_ptr(B_packed, f), nao, naux, _ptr(C_occ, f), nocc, _ptr(D, f), int(s),
                                 _ptr(J, f), _ptr(K, f), _ptr(X_out, f) if X_out is not None else None,
                                 _ptr(e6_out, torch.int32) if e6_out is not None else None,
                                 C.byref(ng), _stream(stream)), "df_debug_jk_build")
    return int(ng.value)


def df_debug_set_gemm_flags(flags: int) -> None:
    _check(lib.df_debug_set_gemm_flags(int(flags)), "df_debug_set_gemm_flags")


def df_launch_count() -> int:
    return int(lib.df_launch_count())


def df_profile_enable(on: bool) -> None:
    _check(lib.df_profile_enable(1 if on else 0), "df_profile_enable")


def df_profile_read() -> dict:
    """{class name: (milliseconds, brackets)} since the last read; synchronises."""
    n = int(lib.df_profile_num_classes())
    ms = (C.c_float * n)()
    cnt = (C.c_int * n)()
    _check(lib.df_profile_read(ms, cnt), "df_profile_read")
    return {lib.df_profile_class_name(i).decode(): (float(ms[i]), int(cnt[i])) for i in range(n)}


def df_debug_mma_peak(n_mma: int, iters: int, grid: int, stream=None) -> float:
    ms = C.c_float(0.0)
    _check(lib.df_debug_mma_peak(int(n_mma), int(iters), int(grid), C.byref(ms), _stream(stream)),
           "df_debug_mma_peak")
    return float(ms.value)
