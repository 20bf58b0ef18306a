"""df_emul_gemm_static: the emulated GEMM for callers that cannot allocate device memory.

Who that is (include/df_emul.h has the full contract): an SCF driver whose HBM is all committed at
start-up, a callback running while its stream is being captured (cudaMalloc is forbidden there), a host
thread beside other contexts' builds that a cudaMalloc would stall by synchronising the device.  They
cannot register a workspace, so this entry point keeps its scratch in a 64 MiB array inside the library.

What is checked: on calls made one after the other, which share that array and find the previous
call's digit planes and column maxima in it, C equals the existing path's C (df_emul_gemm with a
registered workspace) bit for bit -- the comparison the other emulated-GEMM parity tests use -- and is
within `tol` of the oracle's plain FP64 product; a problem beyond the limit is refused with
DF_ERR_TOO_LARGE and C untouched; a call allocates no device memory.

This file is collected last on purpose (pytest -x stops at the first failure, and a failure in this
out-of-scope entry point must not hide a parity test); it passes alone in a fresh process as well as
after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import df_inputs as G
from oracle import df_oracle as O

pytestmark = pytest.mark.gpu
DEV = "cuda"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def test_static_scratch_limit_is_the_documented_one(dfe):
    assert dfe.df_emul_gemm_static_scratch_bytes() == 64 << 20
    # the examples of include/df_emul.h: 2048^3 fits up to s = 7, 1024 x 1024 x 3000 at s = 8
    assert dfe.df_emul_gemm_workspace_bytes(2048, 2048, 2048, 7) <= 64 << 20 < dfe.df_emul_gemm_workspace_bytes(2048, 2048, 2048, 8)
    assert dfe.df_emul_gemm_workspace_bytes(1024, 1024, 3000, 8) <= 64 << 20


def test_emul_gemm_static_matches_workspace_path_on_consecutive_calls(dfe, gpu_ws):
    # (m, n, k, tol, seed).  The second call is smaller than the first, so every byte of scratch it uses
    # holds the first call's planes, scale indices and column maxima when it starts; the column scale
    # of a call that did not clear the maxima would be the larger one left by the call before (the
    # inputs of the first call are scaled up for that).  The third repeats the first shape with new
    # data (the same kernels, all loaded by then: the free-memory check below), the fourth and fifth
    # take other slice counts.
    calls = [(700, 520, 1500, 1e-8, 41, 1e6), (300, 200, 1000, 1e-8, 42, 1.0), (700, 520, 1500, 1e-8, 43, 1e-3),
             (700, 520, 1500, 1e-5, 44, 1.0), (37, 131, 200, 1e-12, 45, 1.0)]
    inputs = []
    for m, n, k, tol, seed, scale in calls:
        A, B = G.make_gemm_inputs(m, n, k, seed=seed)
        A, B = A * scale, B * scale
        inputs.append((A, B, dev(A), dev(B), torch.full((m, n), -7.0, dtype=torch.float64, device=DEV),
                       torch.full((m, n), 7.0, dtype=torch.float64, device=DEV)))
    torch.cuda.synchronize()
    free = []
    for (m, n, k, tol, _, _), (A, B, Ad, Bd, C_static, C_ws) in zip(calls, inputs):
        dfe.df_emul_gemm_static(Ad, Bd, C_static, m, n, k, tol)
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])
    for (m, n, k, tol, _, _), (A, B, Ad, Bd, C_static, C_ws) in zip(calls, inputs):
        dfe.df_emul_gemm(Ad, Bd, C_ws, m, n, k, tol)  # the existing path, caller-allocated workspace
        torch.cuda.synchronize()
        assert torch.equal(C_static, C_ws), (m, n, k, tol)
        err = O.rel_frobenius(C_static.cpu().numpy(), O.gemm_plain(A, B))
        assert err <= tol, (err, tol)
    # the third call repeats the first call's shape and slice count: every kernel it launches was loaded before, so
    # the device's free memory must not have moved across it
    assert free[2] == free[1], free


def test_emul_gemm_static_back_to_back_without_host_sync(dfe, gpu_ws):
    """Two calls enqueued on one stream with no synchronisation in between are ordered by the stream:
    the second must not disturb the first's result."""
    shapes = [(512, 384, 2048, 1e-6, 51), (200, 250, 520, 1e-10, 52)]
    data = []
    for m, n, k, tol, seed in shapes:
        A, B = G.make_gemm_inputs(m, n, k, seed=seed)
        data.append((dev(A), dev(B), torch.empty((m, n), dtype=torch.float64, device=DEV),
                     torch.empty((m, n), dtype=torch.float64, device=DEV)))
    for (m, n, k, tol, _), (Ad, Bd, C_static, _) in zip(shapes, data):
        dfe.df_emul_gemm_static(Ad, Bd, C_static, m, n, k, tol)
    torch.cuda.synchronize()
    for (m, n, k, tol, _), (Ad, Bd, C_static, C_ws) in zip(shapes, data):
        dfe.df_emul_gemm(Ad, Bd, C_ws, m, n, k, tol)
        torch.cuda.synchronize()
        assert torch.equal(C_static, C_ws), (m, n, k, tol)


def test_emul_gemm_static_refuses_what_does_not_fit(dfe, gpu_ws):
    m = n = k = 2048
    tol = 1e-15  # s = 8: 8 * 4096 * 2048 bytes of planes = 64 MiB, plus scale indices: just over
    assert dfe.df_emul_gemm_workspace_bytes(m, n, k, dfe.df_slices_for_tol(tol)) > dfe.df_emul_gemm_static_scratch_bytes()
    A = torch.ones((m, k), dtype=torch.float64, device=DEV)
    B = torch.ones((k, n), dtype=torch.float64, device=DEV)
    C = torch.full((m, n), 3.0, dtype=torch.float64, device=DEV)
    with pytest.raises(dfe.DFError) as ei:
        dfe.df_emul_gemm_static(A, B, C, m, n, k, tol)
    assert ei.value.code == -8 and "DF_ERR_TOO_LARGE" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((C == 3.0).all())
    # the same sizes with fewer slices fit and run
    dfe.df_emul_gemm_static(A, B, C, m, n, k, 1e-6)
    torch.cuda.synchronize()
    assert bool((C == float(k)).all())
    with pytest.raises(dfe.DFError):
        dfe.df_emul_gemm_static(A, B, C, 0, n, k, 1e-6)
