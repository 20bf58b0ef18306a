"""Seeded generators for the synthetic DF workloads (BASELINE.json `configs`).

Recipes (stated again in DESIGN.md "Input recipe"):

* B^q_ij, packed lower-triangular, shape (npair, naux), q fastest,
  p(i, j) = i(i+1)/2 + j for i >= j.  Entries = sign * 10^u, u ~ U(-8, 0) real,
  times a per-q decay exp(-q / naux)                      (configs 0, 2, 3, 4).
* Screened variant: the same entries times exp(-decay |i - j|) (a Schwarz-like fall-off away from
  the diagonal)                               (screening tests, bench --screen).
* C_occ = first nocc columns of the Q factor of a Gaussian nao x nao matrix,
  D = 2 C_occ C_occ^T                                      (configs 0, 2, 3, 4).
* GEMM sweep: entries sign * 2^e, e ~ U(-30, 0) REAL, plus an
  integer per-row offset in [-10, 10] applied to the rows of A and of B
                                                            (config 1).
* SCF sequence: D_k = D* + eps_k S_k, eps_k = 10^(-k/2), S_k random symmetric
  with unit Frobenius norm; C_k from the nocc largest eigenpairs of D_k
                                                (configs 2, 3).

Nothing here belongs to the method: these are inputs only.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class DFConfig:
    name: str
    nao: int
    naux: int
    nocc: int
    seed: int


# BASELINE.json configs 0, 2, 3, 4 (config 1 is the square GEMM sweep).
CONFIGS = {
    "tiny": DFConfig("tiny", 48, 160, 10, 0),
    "medium": DFConfig("medium", 500, 1700, 50, 1),
    "large": DFConfig("large", 1200, 4000, 150, 2),
    "largest": DFConfig("largest", 1800, 6000, 250, 3),
}


def npair(nao: int) -> int:
    return nao * (nao + 1) // 2


def pair_index(i, j):
    """Packed index of the pair (i, j); symmetric in its arguments."""
    i = np.asarray(i)
    j = np.asarray(j)
    hi = np.maximum(i, j)
    lo = np.minimum(i, j)
    return hi * (hi + 1) // 2 + lo


def make_B_packed(nao: int, naux: int, seed: int, dtype=np.float64) -> np.ndarray:
    """(npair, naux) float64, C-contiguous (q fastest)."""
    rng = np.random.default_rng(seed)
    n = npair(nao)
    u = rng.uniform(-8.0, 0.0, size=(n, naux))
    sign = rng.integers(0, 2, size=(n, naux)) * 2 - 1
    decay = np.exp(-np.arange(naux, dtype=np.float64) / naux)
    B = sign * np.power(10.0, u) * decay[None, :]
    return np.ascontiguousarray(B, dtype=dtype)


def make_B_packed_screened(nao: int, naux: int, seed: int, decay: float = 0.25) -> np.ndarray:
    """Packed B with a Schwarz-like decay away from the diagonal: the entries of make_B_packed times
    exp(-decay |i - j|), the shape a screened three-index tensor of a spatially extended molecule
    has (the significant pairs number N_scr <= N_bf^2, normally O(N_bf)).  Far from the
    diagonal the values fall below every slice of their row's scale, so whole blocks of digits are
    zero."""
    B = make_B_packed(nao, naux, seed)
    il, jl = np.tril_indices(nao)
    B *= np.exp(-decay * (il - jl))[:, None]
    return np.ascontiguousarray(B)


def make_C_occ(nao: int, nocc: int, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed + 1000003)
    G = rng.standard_normal((nao, nao))
    Q, _ = np.linalg.qr(G)
    return np.ascontiguousarray(Q[:, :nocc])


def make_density(C_occ: np.ndarray) -> np.ndarray:
    D = 2.0 * (C_occ @ C_occ.T)
    return np.ascontiguousarray(0.5 * (D + D.T))


def make_df_inputs(cfg: DFConfig):
    """(B_packed, C_occ, D) for a DFConfig, all host float64."""
    B = make_B_packed(cfg.nao, cfg.naux, cfg.seed)
    C = make_C_occ(cfg.nao, cfg.nocc, cfg.seed)
    D = make_density(C)
    return B, C, D


def make_gemm_inputs(m: int, n: int, k: int, seed: int):
    """Config-1 style operands A (m x k) and B (k x n), row-major float64."""
    rng = np.random.default_rng(seed)

    def one(rows, cols):
        e = rng.uniform(-30.0, 0.0, size=(rows, cols))
        sign = rng.integers(0, 2, size=(rows, cols)) * 2 - 1
        off = rng.integers(-10, 11, size=(rows, 1)).astype(np.float64)
        return np.ascontiguousarray(sign * np.exp2(e + off))

    return one(m, k), one(k, n)


def make_gemm_inputs_torch(m: int, n: int, k: int, seed: int, device="cuda"):
    """make_gemm_inputs generated on the device for the sizes too large for host time (8192, 16384):
    the same distribution (sign 2^e, real e ~ Uniform(-30, 0), integer per-row offsets in [-10, 10]),
    NOT the same bytes -- a consumer on the host reads these bytes back, it never regenerates them."""
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)

    def one(rows, cols):
        e = torch.rand((rows, cols), generator=g, dtype=torch.float64, device=device) * 30.0 - 30.0
        off = torch.randint(-10, 11, (rows, 1), generator=g, device=device).to(torch.float64)
        sgn = torch.where(torch.rand((rows, cols), generator=g, device=device) < 0.5, -1.0, 1.0).to(torch.float64)
        return sgn * torch.exp2(e + off)

    return one(m, k), one(k, n)


def occ_from_density(D: np.ndarray, nocc: int) -> np.ndarray:
    """C with D ~= 2 C C^T from the nocc largest eigenpairs."""
    lam, V = np.linalg.eigh(0.5 * (D + D.T))
    lam = lam[-nocc:]
    V = V[:, -nocc:]
    return np.ascontiguousarray(V * np.sqrt(np.maximum(lam, 0.0) / 2.0)[None, :])


def make_scf_sequence(D_star: np.ndarray, nocc: int, nsteps: int, seed: int):
    """List of (eps_k, D_k, C_k) for k = 0..nsteps-1."""
    rng = np.random.default_rng(seed + 7777)
    nao = D_star.shape[0]
    out = []
    for k in range(nsteps):
        S = rng.standard_normal((nao, nao))
        S = 0.5 * (S + S.T)
        S /= np.linalg.norm(S)
        eps = 10.0 ** (-k / 2.0)
        Dk = D_star + eps * S
        Dk = np.ascontiguousarray(0.5 * (Dk + Dk.T))
        out.append((eps, Dk, occ_from_density(Dk, nocc)))
    return out


def make_B_packed_torch(nao: int, naux: int, seed: int, device="cuda", chunk_pairs: int = 1 << 16,
                        offdiag_decay: float = 0.0):
    """Device-side generation of packed B for the configs too large for host
    RAM/time (configs 3, 4).  Same distribution as make_B_packed; NOT the same
    bytes (a different generator) -- the oracle always reads these bytes back,
    it never regenerates them.  offdiag_decay > 0: the screened variant,
    entries times exp(-offdiag_decay |i - j|) (make_B_packed_screened)."""
    import torch

    n = npair(nao)
    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    B = torch.empty((n, naux), dtype=torch.float64, device=device)
    decay = torch.exp(-torch.arange(naux, dtype=torch.float64, device=device) / naux)
    ln10 = float(np.log(10.0))
    for p0 in range(0, n, chunk_pairs):
        p1 = min(n, p0 + chunk_pairs)
        u = torch.rand((p1 - p0, naux), generator=gen, dtype=torch.float64, device=device)
        sgn = torch.rand((p1 - p0, naux), generator=gen, dtype=torch.float32, device=device)
        blk = torch.exp(u.mul_(8.0 * ln10).sub_(8.0 * ln10))
        blk.mul_(decay[None, :])
        blk = torch.where(sgn < 0.5, -blk, blk)
        if offdiag_decay > 0.0:
            pidx = torch.arange(p0, p1, dtype=torch.float64, device=device)
            i = torch.floor((torch.sqrt(8.0 * pidx + 1.0) - 1.0) * 0.5)
            i = torch.where(i * (i + 1) / 2 > pidx, i - 1, i)
            i = torch.where((i + 1) * (i + 2) / 2 <= pidx, i + 1, i)
            j = pidx - i * (i + 1) / 2
            blk.mul_(torch.exp(-offdiag_decay * (i - j))[:, None])
        B[p0:p1].copy_(blk)
        del u, sgn, blk
    return B
