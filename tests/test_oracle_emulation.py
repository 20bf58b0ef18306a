"""Pins for oracle part O2 (INT8 slice emulation) -- CPU only.

Each pin is something other than the oracle's own formula: exact identities in
Python integers, an independently derived closed form of the balanced digits,
exact integer matmul on few-digit inputs, and error levels against an
extended-precision product.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle as O
from df_inputs import CONFIGS, make_df_inputs, make_gemm_inputs


def _edge_values():
    vals = [0.0, 1.0, -1.0, 0.5, -0.5, 127.0 / 128.0, -127.0 / 128.0,
            np.nextafter(127.0 / 128.0, 0.0), np.nextafter(127.0 / 128.0, 1.0),
            np.nextafter(1.0, 0.0), 2.0 ** -30, -(2.0 ** -30), 3.0e-11, 1e-300, -1e-300,
            5e-324, 1.7976931348623157e308, 2.0 ** -1000, 2.0 ** -1001, 0.75, -0.3,
            2.0 ** -52, 1 - 2.0 ** -53, 255.0 / 256.0, 0.49609375]
    return np.array(vals)


# ------------------------------------------------------------------ step 1-2


def test_scale_index_headroom_random_and_edges():
    rng = np.random.default_rng(0)
    m = np.concatenate([np.abs(_edge_values()), np.exp2(rng.uniform(-900, 900, 20000)),
                        rng.uniform(0.5, 1.0, 20000), 1.0 - np.exp2(rng.uniform(-20, -6, 2000))])
    e = O.scale_index(m)
    nz = m >= 2.0 ** -1000
    # headroom the balanced digits need: m 2^-e < 127/128, and e is the smallest such
    scaled = np.array([Fraction(float(x)) / Fraction(2) ** int(ee) for x, ee in zip(m[nz][:3000], e[nz][:3000])])
    assert all(v < Fraction(127, 128) for v in scaled)
    assert all(v >= Fraction(127, 256) for v in scaled)
    assert np.all(e[~nz] == 0)


def test_scale_index_boundary_is_top_mantissa_bits():
    # f >= 127/128 <=> hidden bit and the top 6 stored mantissa bits all ones
    for E in (-40, 0, 3, 200):
        for f, bump in ((127.0 / 128.0, 1), (np.nextafter(127.0 / 128.0, 0), 0), (0.5, 0), (np.nextafter(1.0, 0), 1)):
            m = math.ldexp(f, E)
            bits = np.array([m]).view(np.uint64)[0]
            top6 = (int(bits) >> 46) & 63
            assert (top6 == 63) == bool(bump)
            assert int(O.scale_index(np.array([m]))[0]) == E + bump


def test_fixed_point_exact_against_fractions():
    rng = np.random.default_rng(1)
    x = np.concatenate([rng.standard_normal(300) * np.exp2(rng.integers(-60, 5, 300)), _edge_values()[:13]])
    for row in (x[:100], x[100:200], x[200:]):
        m = np.max(np.abs(row))
        e = int(O.scale_index(np.array([m]))[0])
        Q = O.fixed_point(row, np.array(e))
        for xv, q in zip(row, Q):
            exact = Fraction(float(xv)) * Fraction(2) ** (63 - e)
            # round half to even on the exact rational
            fl = exact.numerator // exact.denominator
            rem = exact - fl
            if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and fl % 2 == 1):
                fl += 1
            assert int(q) == fl
            assert abs(int(q)) < (127 * 2 ** 63) // 128 + 1


# ------------------------------------------------------------------ step 3


def _closed_form_digits(Q):
    """Independent derivation: adding 128 at each of the 7 low byte positions
    (carries propagate by themselves) and subtracting it again digit-wise gives
    the unique representation with digits in [-128, 127]."""
    out = []
    for q in Q:
        qp = int(q) + 0x0080808080808080
        assert -(2 ** 63) <= qp < 2 ** 63
        ds = []
        for t in range(1, 9):
            sh = 8 * (8 - t)
            if t == 1:
                ds.append(qp >> 56)  # Python ints: arithmetic shift
            else:
                ds.append(((qp >> sh) & 255) - 128)
        out.append(ds)
    return np.array(out, dtype=np.int64).T


def _random_Q(rng, n):
    lim = (127 * 2 ** 63) // 128
    q = rng.integers(-lim, lim, size=n, dtype=np.int64)
    edges = np.array([0, 1, -1, 127, 128, -128, -129, 255, 256, 32767, 32768, -32768, -32769,
                      lim - 1, -lim + 1, 0x007f7f7f7f7f7f7f, 0x0080808080808080, -0x0080808080808080,
                      0x7e7f7f7f7f7f7f7f, 2 ** 55, -(2 ** 55), 2 ** 56 - 1], dtype=np.int64)
    return np.concatenate([q, edges])


def test_digits_identity_range_and_closed_form():
    rng = np.random.default_rng(2)
    Q = _random_Q(rng, 5000)
    d = O.balanced_digits(Q).astype(np.int64)
    assert d.min() >= -128 and d.max() <= 127
    for col in range(0, Q.size, 7):
        assert sum(int(d[t, col]) * 256 ** (7 - t) for t in range(8)) == int(Q[col])
    assert np.array_equal(d, _closed_form_digits(Q))


def test_digits_prefix_property():
    rng = np.random.default_rng(3)
    Q = _random_Q(rng, 3000)
    d = O.balanced_digits(Q).astype(np.int64)
    for s in range(1, 8):
        unit = 256 ** (8 - s)
        for col in range(0, Q.size, 11):
            prefix = sum(int(d[t, col]) * 256 ** (7 - t) for t in range(s))
            assert prefix % unit == 0
            # tail of balanced digits: within 128/255 of one unit of slice s
            assert abs(int(Q[col]) - prefix) * 255 <= 128 * unit
    # digits do not depend on s: split_operand(s) is a prefix of split_operand(8)
    X = rng.standard_normal((5, 33)) * np.exp2(rng.integers(-20, 3, (5, 33)))
    e8, D8 = O.split_operand(X, 8)
    for s in (1, 3, 6):
        es, Ds = O.split_operand(X, s)
        assert np.array_equal(es, e8) and np.array_equal(Ds, D8[:s])


def test_split_reconstructs_value():
    rng = np.random.default_rng(4)
    X = rng.standard_normal((6, 40)) * np.exp2(rng.integers(-9, 1, (6, 40)))
    e, Dg = O.split_operand(X, 8)
    for i in range(6):
        for k in range(0, 40, 3):
            val = sum(Fraction(int(Dg[t, i, k])) * Fraction(2) ** (1 - 8 * (t + 1)) for t in range(8))
            val *= Fraction(2) ** int(e[i])
            # all elements within 2^-10 of the row max are captured exactly (63-bit Q)
            if abs(X[i, k]) >= 2.0 ** (int(e[i]) - 10):
                assert val == Fraction(float(X[i, k]))
            else:
                assert abs(val - Fraction(float(X[i, k]))) <= Fraction(2) ** (int(e[i]) - 64)


def test_zero_and_tiny_rows():
    X = np.array([[0.0, 0.0, 0.0], [1e-310, -2e-305, 0.0], [2.0 ** -1000, 0.0, 2.0 ** -1001]])
    e, Dg = O.split_operand(X, 8)
    assert e[0] == 0 and e[1] == 0 and not Dg[:, :2].any()
    assert e[2] == -999 and Dg[0, 2, 0] == 64 and Dg[0, 2, 2] == 32


# ------------------------------------------------------------------ step 4


def test_pair_products_exact_identity_all_pairs():
    rng = np.random.default_rng(5)
    A = rng.standard_normal((4, 9)) * np.exp2(rng.integers(-12, 2, (4, 9)))
    B = rng.standard_normal((9, 3)) * np.exp2(rng.integers(-12, 2, (9, 3)))
    eA, DA = O.split_operand(A, 8)
    eB, DB = O.split_operand(B.T.copy(), 8)
    QA = O.fixed_point(A, eA[:, None])
    QB = O.fixed_point(B.T.copy(), eB[:, None])
    for i in range(4):
        for j in range(3):
            exact = sum(int(QA[i, k]) * int(QB[j, k]) for k in range(9))
            tot = 0
            for t in range(1, 9):
                for u in range(1, 9):
                    P = O.pair_product(DA[t - 1], DB[u - 1])
                    tot += int(P[i, j]) * 256 ** (16 - t - u)
            assert tot == exact


def test_pair_product_float_shortcut_equals_int64():
    rng = np.random.default_rng(6)
    DA = rng.integers(-128, 128, (37, 515)).astype(np.int8)
    DB = rng.integers(-128, 128, (29, 515)).astype(np.int8)
    DA[0, :] = -128
    DB[0, :] = -128
    assert np.array_equal(O.pair_product(DA, DB), O.pair_product_int64(DA, DB))
    assert O.pair_product(DA, DB)[0, 0] == 515 * 16384


def test_weight_sums_count_and_membership():
    rng = np.random.default_rng(7)
    DA = rng.integers(-128, 128, (8, 5, 16)).astype(np.int8)
    DB = rng.integers(-128, 128, (8, 6, 16)).astype(np.int8)
    for s in range(1, 9):
        Pw = O.weight_sums(DA, DB, s)
        assert sorted(Pw) == list(range(2, s + 2))
        npairs = 0
        for w in Pw:
            ref = np.zeros((5, 6), dtype=np.int64)
            for t in range(1, s + 1):
                for u in range(1, s + 1):
                    if t + u == w:
                        ref += DA[t - 1].astype(np.int64) @ DB[u - 1].astype(np.int64).T
                        npairs += 1
            assert np.array_equal(Pw[w], ref)
        assert npairs == s * (s + 1) // 2 == O.num_int8_gemms(s)


def test_kflush_guard():
    for s in range(1, 9):
        kf = O.kflush(s)
        assert kf % 32 == 0 and s * kf <= 131071 < s * (kf + 32)
        # worst case |P^(w)| <= (#pairs of one weight <= s) * k * 2^14 < 2^31
        assert s * kf * (1 << 14) < (1 << 31)
    assert O.kflush(8) == 16352


# ------------------------------------------------------------------ steps 5-6


def test_recombination_order_term_by_term():
    """The flat running sum (reading R6) re-derived with Python floats."""
    rng = np.random.default_rng(8)
    A = rng.standard_normal((3, 70)) * np.exp2(rng.integers(-8, 1, (3, 70)))
    B = rng.standard_normal((70, 2))
    s = 4
    eA, DA = O.split_operand(A, s)
    eB, DB = O.split_operand(B.T.copy(), s)
    C = O.emul_gemm(A, B, s)
    for i in range(3):
        for j in range(2):
            acc = 0.0
            for w in range(s + 1, 1, -1):
                P = 0
                for t in range(1, s + 1):
                    u = w - t
                    if 1 <= u <= s:
                        P += sum(int(DA[t - 1, i, k]) * int(DB[u - 1, j, k]) for k in range(70))
                acc = acc + math.ldexp(float(P), int(eA[i] + eB[j]) + 2 - 8 * w)
            assert acc == C[i, j]


def test_chunked_flush_matches_manual(monkeypatch):
    """With a tiny KFLUSH the chunks are added in increasing-k order."""
    rng = np.random.default_rng(9)
    A = rng.standard_normal((4, 100))
    B = rng.standard_normal((100, 5))
    s = 3
    monkeypatch.setattr(O.df_oracle, "kflush", lambda s_: 32)
    C = O.df_oracle.emul_gemm(A, B, s)
    eA, DA = O.split_operand(A, s)
    eB, DB = O.split_operand(B.T.copy(), s)
    ref = np.zeros((4, 5))
    for k0 in range(0, 100, 32):
        Pw = O.weight_sums(DA, DB, s, k0, min(100, k0 + 32))
        for w in range(s + 1, 1, -1):
            ref = ref + np.ldexp(Pw[w].astype(np.float64), (eA[:, None] + eB[None, :] + 2 - 8 * w).astype(np.int32))
    assert np.array_equal(C, ref)


@pytest.mark.parametrize("digits,s", [(1, 1), (2, 3), (3, 5), (4, 7)])
def test_exact_on_few_digit_integers(digits, s):
    """Inputs with `digits` nonzero base-256 digits and s >= 2*digits-1 keep
    every nonzero pair, so the emulation IS the exact integer product."""
    rng = np.random.default_rng(10 + digits)
    m, k, n = 13, 300, 11
    lim = 100 * 256 ** (digits - 1)
    A = rng.integers(-lim, lim + 1, (m, k)).astype(np.float64)
    B = rng.integers(-lim, lim + 1, (k, n)).astype(np.float64)
    # pin every row/column max to 100 * 256^(digits-1): Q = x 2^(64 - 8 digits)
    A[:, 0] = lim
    B[0, :] = -lim
    C = O.emul_gemm(A, B, s)
    exact = A.astype(np.int64).astype(object) @ B.astype(np.int64).astype(object)
    big = max(abs(int(v)) for v in exact.ravel())
    if big < 2 ** 53:
        assert np.array_equal(C, exact.astype(np.float64))
    else:
        # the exact integer no longer fits FP64: each of the s weight additions rounds once
        for c, ex in zip(C.ravel(), exact.ravel()):
            assert abs(Fraction(float(c)) - ex) <= s * Fraction(math.ulp(float(big)))
    if s > 1:  # dropping the last weight must break exactness (a dropped-term mistake fails)
        Cm = O.emul_gemm(A, B, s - 1)
        errs = [abs(Fraction(float(c)) - ex) for c, ex in zip(Cm.ravel(), exact.ravel())]
        assert max(errs) > 2 * s * Fraction(math.ulp(float(big)))


def test_power_of_two_scaling_commutes():
    """Scaling a row of A / column of B by 2^p scales C's row / column exactly."""
    rng = np.random.default_rng(21)
    A = rng.standard_normal((6, 50))
    B = rng.standard_normal((50, 7))
    C = O.emul_gemm(A, B, 4)
    A2 = A.copy(); A2[2] *= 2.0 ** 17
    B2 = B.copy(); B2[:, 3] *= 2.0 ** -9
    C2 = O.emul_gemm(A2, B2, 4)
    ref = C.copy(); ref[2] *= 2.0 ** 17; ref[:, 3] *= 2.0 ** -9
    assert np.array_equal(C2, ref)


def test_transposed_operand_mistake_detected():
    rng = np.random.default_rng(22)
    A = rng.standard_normal((8, 8))
    B = rng.standard_normal((8, 8))
    C = O.emul_gemm(A, B, 6)
    assert O.rel_frobenius(C, A @ B) < 1e-12
    assert O.rel_frobenius(C, A @ B.T) > 0.1


@pytest.mark.parametrize("tol", [1e-4, 1e-6, 1e-8, 1e-10, 1e-12])
def test_error_within_tol_on_config1_like_data(tol):
    A, B = make_gemm_inputs(96, 80, 640, seed=3)
    ref = O.gemm_longdouble(A, B)
    s = O.slices_for_tol(tol, "guarded")
    err = O.rel_frobenius(O.emul_gemm(A, B, s).astype(np.longdouble), ref)
    assert err <= tol
    # error shrinks by ~2^8 per slice until FP64 round-off
    if s >= 2:
        err_m = O.rel_frobenius(O.emul_gemm(A, B, s - 1).astype(np.longdouble), ref)
        assert err_m > 20 * err or err < 1e-15


def test_max_slices_below_1e12_vs_plain():
    A, B = make_gemm_inputs(64, 64, 512, seed=4)
    assert O.rel_frobenius(O.emul_gemm(A, B, 8), O.gemm_plain(A, B)) <= 1e-12


# ------------------------------------------------------------------ step 7 (K path)


def test_q_groups_rule_and_int32_guard():
    """Reading R5 / SURVEY 8(c) step 7, stated without the oracle's formula: the groups partition
    [0, naux) in order, never straddle a q-block, are as long as the INT32 guard allows, and the worst
    case of one weight sum over a group (s pairs, every digit -128: s |g| nocc 2^14) stays below 2^31."""
    for naux, nocc, s, qb in [(160, 10, 3, 512), (1700, 50, 8, 512), (4000, 150, 4, 512), (4000, 150, 6, 512),
                              (6000, 250, 5, 512), (37, 250, 8, 16), (1300, 70, 4, 512), (700, 1, 1, 512)]:
        g = O.q_groups(naux, nocc, s, qb)
        assert g[0][0] == 0 and g[-1][1] == naux
        for (a0, a1), (b0, b1) in zip(g[:-1], g[1:]):
            assert a1 == b0 and a0 < a1
        for g0, g1 in g:
            n = g1 - g0
            assert g0 // qb == (g1 - 1) // qb  # never straddles a q-block
            assert s * n * nocc * (1 << 14) < (1 << 31)  # INT32 guard, true worst case
            last_of_block = g1 == naux or g1 % qb == 0
            if not last_of_block:
                # maximal: one more q would exceed the flush length (a multiple of the 32-byte MMA K)
                k_allowed = 32 * (((1 << 17) - 1) // (32 * s))
                assert (n + 1) * nocc > k_allowed
    # the configuration the benchmark runs (PAPER.md:200-222 shapes): 512 = 218 + 218 + 76 at s = 4
    assert O.q_groups(4000, 150, 4)[:3] == [(0, 218), (218, 436), (436, 512)]


def test_k_path_exact_on_small_integers():
    """1-digit integer B and C: X is an exact integer with <= 3 digits at s >= 3;
    K = X X^T is exact at s = 5.  Pins the whole K path (unpack, GEMM(5),
    per-group re-split, GEMM(6), group sum)."""
    rng = np.random.default_rng(31)
    nao, naux, nocc = 12, 9, 4
    Bp = rng.integers(-100, 101, (O.npair(nao), naux)).astype(np.float64)
    C = rng.integers(-100, 101, (nao, nocc)).astype(np.float64)
    # pin all scales: every unpacked row of every B^q and every column of C has max 100
    for i in range(nao):
        Bp[i * (i + 1) // 2 + i, :] = 100.0
    C[0, :] = 100.0
    K, X = O.emul_df_k(Bp, nao, C, 5, qblock=4, return_x=True)
    Xe = np.empty((naux, nao, nocc), dtype=object)
    Ke = np.zeros((nao, nao), dtype=object)
    Ci = C.astype(np.int64).astype(object)
    for q in range(naux):
        Bq = O.unpack_sym(Bp[:, q], nao).astype(np.int64).astype(object)
        Xe[q] = Bq @ Ci
        Ke += Xe[q] @ Xe[q].T
    assert np.array_equal(X, Xe.astype(np.float64))
    assert np.array_equal(K, Ke.astype(np.float64))


@pytest.mark.parametrize("tol", [1e-4, 1e-8, 1e-12])
def test_k_path_within_tol_on_tiny_config(tol):
    cfg = CONFIGS["tiny"]
    Bp, C, D = make_df_inputs(cfg)
    J, K = O.df_jk_plain(Bp, cfg.nao, C, D)
    s = O.slices_for_tol(tol)
    Je, Ke = O.emul_df_jk(Bp, cfg.nao, C, D, s, qblock=64)
    assert np.array_equal(Je, J)  # J is plain FP64
    assert np.array_equal(Ke, Ke.T)
    assert O.rel_frobenius(Ke, K) <= tol
    lam = np.linalg.eigvalsh(Ke)
    assert lam.min() > -tol * lam.max()


def test_k_path_max_slices():
    cfg = CONFIGS["tiny"]
    Bp, C, D = make_df_inputs(cfg)
    K = O.df_k(Bp, cfg.nao, C)
    assert O.rel_frobenius(O.emul_df_k(Bp, cfg.nao, C, 8), K) <= 1e-12


def test_level0_emulation_is_at_least_fp64_accurate():
    """Table 1's level 0 is "standard FP64", relative accuracy 2.2e-16.  The library
    has no native-FP64 GEMM: the caller-side schedule passes tol = 2^-52 and the guarded policy turns
    that into s = 8.  Pin what that delivers against an extended-precision reference (x86 long double,
    64-bit mantissa): on the config-1-like GEMM data and on the config-0 K path the s = 8 emulation is
    closer to the exact result than the plain FP64 evaluation itself, and within 2.2e-16."""
    assert O.slices_for_tol(2.0 ** -52, "guarded") == 8
    A, B = make_gemm_inputs(96, 80, 640, seed=3)
    ref = O.gemm_longdouble(A, B)
    e_emul = O.rel_frobenius(O.emul_gemm(A, B, 8).astype(np.longdouble), ref)
    e_fp64 = O.rel_frobenius(O.gemm_plain(A, B).astype(np.longdouble), ref)
    assert e_emul <= e_fp64 and e_emul <= 2.0 ** -52, (e_emul, e_fp64)
    cfg = CONFIGS["tiny"]
    Bp, C, D = make_df_inputs(cfg)
    Kl = np.zeros((cfg.nao, cfg.nao), dtype=np.longdouble)
    Cl = C.astype(np.longdouble)
    for q in range(cfg.naux):
        Xq = O.unpack_sym(Bp[:, q], cfg.nao).astype(np.longdouble) @ Cl
        Kl += Xq @ Xq.T
    e_emul = O.rel_frobenius(O.emul_df_k(Bp, cfg.nao, C, 8).astype(np.longdouble), Kl)
    e_fp64 = O.rel_frobenius(O.df_k(Bp, cfg.nao, C).astype(np.longdouble), Kl)
    assert e_emul <= e_fp64 and e_emul <= 2.0 ** -52, (e_emul, e_fp64)


def test_status_bits():
    X = np.ones((3, 4))
    assert O.operand_status(X) == 0
    Y = X.copy(); Y[1, 2] = np.inf
    assert O.operand_status(Y) & 1
    Z = X.copy(); Z[2] *= 2.0 ** 460
    assert O.operand_status(Z) == 2
