"""CPU oracle for the DF J/K hot path of arXiv 2601.08077 -- TEST INFRASTRUCTURE.

This file is test infrastructure, not the product.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import it.  It shares no code with `paper_2601_08077_b200/` (the CUDA
path) and imports nothing from it.  Plain NumPy, FP64 (exact integers in int64 /
Python int), slow and meant to be checked against the paper by eye.

Part O1 -- the plain result (what the method approximates):
    rho_q = sum_ij B^q_ij D_ij                 PAPER.md:45  (Eq. 3, "Y^q")
    J_ij  = sum_q  B^q_ij rho_q                PAPER.md:47  (Eq. 4)
    X^q_ia = sum_j B^q_ij C_ja                 PAPER.md:49-51 (Eq. 5, "W^q_is")
    K_ij  = sum_q sum_a X^q_ia X^q_ja          PAPER.md:53  (Eq. 6)

Part O2 -- the INT8 emulation of an FP64 GEMM, step by step.  The paper gives
only "fixed point emulation ... follows the Ozaki scheme", s = ceil((m+1)/8)
INT8 splits and s(s+1)/2 INT8 GEMMs ("10 or more" at 4 splits,
PAPER.md:139); every further detail is the reading fixed in DESIGN.md
("Readings", R1..R9):

  step 1  scale index e per row of the left / column of the right operand
  step 2  Q = rint(x * 2^(63-e)) as int64
  step 3  balanced base-256 digits d_1..d_8 in [-128, 127], sum d_t 256^(8-t) = Q
  step 4  P^(t,u) = D^A_t . D^B_u (exact integers) for t+u <= s+1,
          P^(w) = sum_{t+u=w} P^(t,u)
  step 5  C = sum over k-chunks (increasing k), within a chunk over
          w = s+1 down to 2 (smallest weight first), of
          2^(eA_i + eB_j + 2 - 8w) * P^(w)_ij  -- ONE running FP64 sum
  step 6  a chunk holds at most KFLUSH(s) = 32*floor(131071/(32 s)) contraction
          elements (INT32 guard s*k < 2^17)
  step 7  K path: GEMM(5) rows (q,i) / contraction j; GEMM(6) rows i /
          contraction (q,a) inside one q-group; scale of X per (i, group)

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): brute-force 4-index
contraction, symmetry/PSD/trace invariants, naux=1 rank-one case, exact digit
identity in Python ints, an independently derived closed form of the balanced
digits, the exact product identity over all 64 pairs, exactness on few-digit
integer inputs (reduces to integer matmul), Table 1 of the paper
(tests/golden/table1_paper.txt).  Unpinned: nothing in this file is "parity
unpinned"; the LAST BITS of the FP64 recombination are fixed only by the
order stated in step 5 (a reading, R6), which the tests pin by re-deriving the
sum term by term in Python floats on a small case.
"""
from __future__ import annotations

import math

import numpy as np

# ----------------------------------------------------------------------------
# packed-pair helpers (data layout of B_packed: BASELINE.json configs[0])
# ----------------------------------------------------------------------------


def npair(nao: int) -> int:
    return nao * (nao + 1) // 2


def unpack_sym(v: np.ndarray, nao: int) -> np.ndarray:
    """Packed lower triangle v[p(i,j)], p = i(i+1)/2 + j (i >= j) -> symmetric nao x nao."""
    M = np.zeros((nao, nao), dtype=v.dtype)
    il, jl = np.tril_indices(nao)  # row-major lower triangle == p order
    M[il, jl] = v
    M[jl, il] = v
    return M


# ----------------------------------------------------------------------------
# Part O1: plain FP64 DF J/K
# ----------------------------------------------------------------------------


def df_rho(B_packed: np.ndarray, nao: int, D: np.ndarray) -> np.ndarray:
    """rho_q = sum_{ij} B^q_ij D_ij  (Eq. 3).  The full sum over
    (i, j) of a symmetric B and symmetric D is the packed sum with weight 1 on
    the diagonal and 2 off it."""
    il, jl = np.tril_indices(nao)
    w = np.where(il == jl, 1.0, 2.0)
    d = 0.5 * (D[il, jl] + D[jl, il])  # D is only read as symmetric
    return (w * d) @ B_packed


def df_j(B_packed: np.ndarray, nao: int, rho: np.ndarray) -> np.ndarray:
    """J_ij = sum_q B^q_ij rho_q  (Eq. 4), full symmetric matrix."""
    return unpack_sym(B_packed @ rho, nao)


def df_x(B_packed: np.ndarray, nao: int, C_occ: np.ndarray) -> np.ndarray:
    """X[q, i, a] = sum_j B^q_ij C_ja  (Eq. 5)."""
    naux = B_packed.shape[1]
    X = np.empty((naux, nao, C_occ.shape[1]))
    for q in range(naux):
        X[q] = unpack_sym(B_packed[:, q], nao) @ C_occ
    return X


def df_k(B_packed: np.ndarray, nao: int, C_occ: np.ndarray) -> np.ndarray:
    """K_ij = sum_q sum_a X^q_ia X^q_ja  (Eq. 6; no occupation
    factor -- reading R8)."""
    K = np.zeros((nao, nao))
    for q in range(B_packed.shape[1]):
        Xq = unpack_sym(B_packed[:, q], nao) @ C_occ
        K += Xq @ Xq.T
    return 0.5 * (K + K.T)


def df_jk_plain(B_packed, nao, C_occ, D):
    """The plain FP64 result of `df_jk_build` (J in FP64: PAPER.md:101)."""
    rho = df_rho(B_packed, nao, D)
    return df_j(B_packed, nao, rho), df_k(B_packed, nao, C_occ)


def gemm_plain(A: np.ndarray, B: np.ndarray) -> np.ndarray:
    """The plain result of `df_emul_gemm`."""
    return A @ B


def gemm_longdouble(A: np.ndarray, B: np.ndarray) -> np.ndarray:
    """A @ B accumulated in extended precision (for checks below FP64 round-off
    of a k-term sum; x86 long double has a 64-bit mantissa)."""
    return (A.astype(np.longdouble) @ B.astype(np.longdouble))


def flops_model(nao: int, naux: int, nocc: int):
    """Effective FLOPs per build, PAPER.md:122-126 with N_scr = N_bf^2:
    J = 4 N_bf^2 N_aux,  K = 2 (N_scr + N_bf^2) N_aux N_occ = 4 N_bf^2 N_aux N_occ."""
    return {"J": 4 * nao * nao * naux, "K": 4 * nao * nao * naux * nocc}


# ----------------------------------------------------------------------------
# Policy: tol -> slices, Table 1 schedule
# ----------------------------------------------------------------------------

# Table 1: threshold lower bound of dE_rel, level, m_emu.
TABLE1 = (
    (2e-6, 4, 23),
    (5e-9, 3, 31),
    (2e-11, 2, 39),
    (7e-14, 1, 47),
)
S_MAX = 8


def slices_from_mantissa_bits(m_emu: int) -> int:
    """s = ceil((m_emu + 1) / 8)."""
    return -(-(m_emu + 1) // 8)


def num_int8_gemms(s: int) -> int:
    """s(s+1)/2 slice-pair products (4 splits <-> 10 GEMMs)."""
    return s * (s + 1) // 2


def slices_for_tol(tol: float, mode: str = "guarded") -> int:
    """tol -> slice count (reading R7).
    nominal: m_emu = ceil(log2(1/tol) - 0.05), s = ceil((m_emu+1)/8)
    guarded: s = ceil((log2(1/tol) + 7) / 8)       (the library default)
    both clamped to 1..8."""
    if not (tol > 0.0) or math.isnan(tol):
        raise ValueError("tol must be positive")
    lg = math.log2(1.0 / tol)
    if mode == "nominal":
        m_emu = max(0, math.ceil(lg - 0.05))
        s = slices_from_mantissa_bits(m_emu)
    elif mode == "guarded":
        s = math.ceil((lg + 7.0) / 8.0)
    else:
        raise ValueError(mode)
    return min(S_MAX, max(1, s))


def table1_level(dE_rel: float):
    """(level, m_emu) for the NEXT iteration from dE_rel of this one
    (PAPER.md:141-147).  Level 0 = native FP64 (m_emu None)."""
    for lo, level, m in TABLE1:
        if dE_rel >= lo:
            return level, m
    return 0, None


def adaptive_schedule(dE_rels):
    """m_emu per SCF iteration: iteration 0 starts at m_emu = 23; iteration i+1
    takes Table 1 on dE_rel_i; never revert to a lower precision
    (PAPER.md:151).  Returns a list of (level, m_emu) of len(dE_rels)+1."""
    out = [(4, 23)]
    cur = 4
    for d in dE_rels:
        level, _ = table1_level(d)
        cur = min(cur, level)  # lower level number == higher precision
        m = {4: 23, 3: 31, 2: 39, 1: 47, 0: None}[cur]
        out.append((cur, m))
    return out


# ----------------------------------------------------------------------------
# Part O2 steps 1-3: scale index, fixed point, balanced digits
# ----------------------------------------------------------------------------

TINY_ROW = 2.0 ** -1000  # rows whose max is below this are zero rows (R9)


def scale_index(m: np.ndarray) -> np.ndarray:
    """Step 1.  m = max |x| over the contraction (>= 0).  m = f 2^E, f in
    [0.5, 1); e = E + 1 if f >= 127/128 else E; zero rows (m < 2^-1000) e = 0.
    Guarantees |x| 2^-e < 127/128."""
    m = np.asarray(m, dtype=np.float64)
    f, E = np.frexp(m)
    e = E.astype(np.int64) + (f >= 127.0 / 128.0)
    return np.where(m < TINY_ROW, 0, e).astype(np.int64)


def fixed_point(x: np.ndarray, e: np.ndarray) -> np.ndarray:
    """Step 2.  Q = round-to-nearest-even(x 2^(63-e)) as int64; `e` broadcasts
    against x.  |Q| < (127/128) 2^63."""
    y = np.ldexp(np.asarray(x, dtype=np.float64), (63 - np.asarray(e)).astype(np.int32))
    return np.rint(y).astype(np.int64)


def balanced_digits(Q: np.ndarray) -> np.ndarray:
    """Step 3.  int8 array of shape (8,) + Q.shape; digits[t-1] = d_t.
    carry chain from the lowest byte up: v = byte_t(Q) + carry; for t > 1,
    v >= 128 -> v -= 256, carry = 1.  byte_1 is the signed top byte."""
    Q = np.asarray(Q, dtype=np.int64)
    d = np.empty((8,) + Q.shape, dtype=np.int64)
    carry = np.zeros(Q.shape, dtype=np.int64)
    for t in range(8, 0, -1):
        if t > 1:
            byte = (Q >> (8 * (8 - t))) & 255
        else:
            byte = Q >> 56  # arithmetic shift: signed top byte
        v = byte + carry
        if t > 1:
            carry = (v >= 128).astype(np.int64)
            v = v - 256 * carry
        d[t - 1] = v
    assert d.min(initial=0) >= -128 and d.max(initial=0) <= 127
    return d.astype(np.int8)


def split_operand(X: np.ndarray, s: int):
    """Rows of X are the vectors that get one scale each (left operand: rows of
    A; right operand: pass B^T so rows = columns of B).  Returns (e, digits)
    with e int64 (rows,) and digits int8 (s, rows, k)."""
    X = np.asarray(X, dtype=np.float64)
    m = np.max(np.abs(X), axis=1) if X.shape[1] else np.zeros(X.shape[0])
    e = scale_index(m)
    Q = fixed_point(X, e[:, None])
    return e, balanced_digits(Q)[:s]


def operand_status(X: np.ndarray) -> int:
    """Data-dependent fault bits the library reports (reading R9):
    bit 0: Inf/NaN present; bit 1: a row max outside [2^-450, 2^450]."""
    X = np.asarray(X, dtype=np.float64)
    st = 0
    if not np.all(np.isfinite(X)):
        st |= 1
    m = np.max(np.abs(X), axis=1)
    m = m[np.isfinite(m) & (m >= TINY_ROW)]
    if m.size and (m.max() >= 2.0 ** 450 or m.min() < 2.0 ** -450):
        st |= 2
    return st


# ----------------------------------------------------------------------------
# Part O2 steps 4-6: slice-pair products, recombination
# ----------------------------------------------------------------------------


def kflush(s: int) -> int:
    """Step 6: largest multiple of 32 with s * k < 2^17."""
    return 32 * (131071 // (32 * s))


def pair_product(DA_t: np.ndarray, DB_u: np.ndarray) -> np.ndarray:
    """P^(t,u) = D^A_t . (D^B_u)^T in exact integers.  float64 BLAS on
    integer-valued matrices is exact while k 2^14 < 2^53; the
    tests check this shortcut against true int64 arithmetic."""
    k = DA_t.shape[1]
    assert k * (1 << 14) < (1 << 53)
    P = DA_t.astype(np.float64) @ DB_u.astype(np.float64).T
    return P.astype(np.int64)


def pair_product_int64(DA_t: np.ndarray, DB_u: np.ndarray) -> np.ndarray:
    return DA_t.astype(np.int64) @ DB_u.astype(np.int64).T


def weight_sums(DA: np.ndarray, DB: np.ndarray, s: int, k0: int = 0, k1: int | None = None):
    """Step 4.  {w: P^(w)} for w = 2..s+1 over contraction range [k0, k1)."""
    out = {}
    for w in range(2, s + 2):
        P = None
        for t in range(1, s + 1):
            u = w - t
            if 1 <= u <= s:
                p = pair_product(DA[t - 1][:, k0:k1], DB[u - 1][:, k0:k1])
                P = p if P is None else P + p
        out[w] = P
    return out


def recombine_into(C: np.ndarray, Pw: dict, s: int, eA: np.ndarray, eB: np.ndarray) -> None:
    """Step 5 for one chunk: C += 2^(eA_i+eB_j+2-8w) P^(w), w = s+1 down to 2,
    one running FP64 sum (each term is exact: an int32-range integer times a
    power of two)."""
    ee = (eA[:, None] + eB[None, :]).astype(np.int64)
    for w in range(s + 1, 1, -1):
        term = np.ldexp(Pw[w].astype(np.float64), (ee + (2 - 8 * w)).astype(np.int32))
        C += term


def emul_gemm_digits(eA, DA, eB, DB, s: int) -> np.ndarray:
    """Steps 4-6 given split operands (DA: (s, m, k), DB: (s, n, k))."""
    m, k = DA.shape[1], DA.shape[2]
    n = DB.shape[1]
    C = np.zeros((m, n))
    kf = kflush(s)
    for k0 in range(0, max(k, 1), kf):
        k1 = min(k, k0 + kf)
        Pw = weight_sums(DA, DB, s, k0, k1)
        for w, P in Pw.items():
            assert np.abs(P).max(initial=0) < (1 << 31), "INT32 guard violated"
        recombine_into(C, Pw, s, eA, eB)
    return C


def emul_gemm(A: np.ndarray, B: np.ndarray, s: int) -> np.ndarray:
    """The emulated FP64 GEMM C = A . B with s INT8 slices (steps 1-6).
    A: m x k, B: k x n."""
    eA, DA = split_operand(A, s)
    eB, DB = split_operand(np.ascontiguousarray(B.T), s)
    return emul_gemm_digits(eA, DA, eB, DB, s)


# ----------------------------------------------------------------------------
# Part O2 step 7: the K path
# ----------------------------------------------------------------------------


def q_groups(naux: int, nocc: int, s: int, qblock: int = 512):
    """Consecutive-q groups for GEMM(6) (reading R5; "a run of
    consecutive q with |g| nocc <= k_flush"): q is cut into blocks of `qblock`; every
    block into runs of at most QG = floor(KFLUSH(s) / nocc) consecutive q, so that the
    |g| nocc contraction elements of one group fit one INT32 chunk (step 6)."""
    qg = max(1, kflush(s) // nocc)
    groups = []
    for b0 in range(0, naux, qblock):
        b1 = min(naux, b0 + qblock)
        for g0 in range(b0, b1, qg):
            groups.append((g0, min(b1, g0 + qg)))
    return groups


def emul_x_group(B_packed, nao, C_occ, s, q0, q1, eC=None, DC=None):
    """GEMM(5) for q in [q0, q1): X[q, i, a], emulated.  Left operand rows
    (q, i) with scale e5[q, i] over the UNPACKED row; right operand C_occ with a
    scale per column a."""
    if eC is None:
        eC, DC = split_operand(np.ascontiguousarray(C_occ.T), s)
    nocc = C_occ.shape[1]
    X = np.empty((q1 - q0, nao, nocc))
    for q in range(q0, q1):
        Bq = unpack_sym(B_packed[:, q], nao)
        e5, D5 = split_operand(Bq, s)
        X[q - q0] = emul_gemm_digits(e5, D5, eC, DC, s)
    return X


def emul_k_from_x_group(Xg: np.ndarray, s: int, K: np.ndarray) -> None:
    """GEMM(6) for one q-group: Xg[q, i, a] -> rows i, contraction (q, a);
    scale per (i, group); K += terms, smallest weight first (flat sum)."""
    nq, nao, nocc = Xg.shape
    Xrow = np.ascontiguousarray(np.transpose(Xg, (1, 0, 2)).reshape(nao, nq * nocc))
    assert Xrow.shape[1] <= kflush(s)
    e6, D6 = split_operand(Xrow, s)
    Pw = weight_sums(D6, D6, s)
    recombine_into(K, Pw, s, e6, e6)


def emul_df_k(B_packed, nao, C_occ, s, qblock: int = 512, return_x: bool = False):
    """Emulated K (step 7): groups added in increasing-q order."""
    naux = B_packed.shape[1]
    nocc = C_occ.shape[1]
    eC, DC = split_operand(np.ascontiguousarray(C_occ.T), s)
    K = np.zeros((nao, nao))
    Xall = np.empty((naux, nao, nocc)) if return_x else None
    for (g0, g1) in q_groups(naux, nocc, s, qblock):
        Xg = emul_x_group(B_packed, nao, C_occ, s, g0, g1, eC, DC)
        if return_x:
            Xall[g0:g1] = Xg
        emul_k_from_x_group(Xg, s, K)
    if return_x:
        return K, Xall
    return K


def emul_df_jk(B_packed, nao, C_occ, D, s, qblock: int = 512):
    """What `df_jk_build` computes: J plain FP64, K emulated."""
    rho = df_rho(B_packed, nao, D)
    return df_j(B_packed, nao, rho), emul_df_k(B_packed, nao, C_occ, s, qblock)


def rel_frobenius(X: np.ndarray, ref: np.ndarray) -> float:
    ref = np.asarray(ref)
    den = float(np.linalg.norm(ref.astype(np.float64)))
    num = float(np.linalg.norm((np.asarray(X) - ref).astype(np.float64)))
    return num / den if den > 0 else num
