"""Pins for oracle part O1 (plain FP64 DF J/K) -- CPU only.

The oracle is checked against things other than itself: an explicit 4-index
tensor (ij|kl) = sum_q B^q_ij B^q_kl built with Python-level loops / einsum on
full (unpacked) arrays, invariants the mathematics fixes, and a rank-one closed
form.  (BASELINE.json north_star; SURVEY.md section 8(c) "What pins each part".)
"""
import numpy as np
import pytest

import oracle as O
from df_inputs import CONFIGS, make_df_inputs, pair_index


def _full_B(Bp, nao):
    """Independent unpack: element-by-element through pair_index (the input
    module's definition of p(i,j)), not oracle.unpack_sym."""
    naux = Bp.shape[1]
    Bf = np.empty((naux, nao, nao))
    for i in range(nao):
        for j in range(nao):
            Bf[:, i, j] = Bp[int(pair_index(i, j))]
    return Bf


@pytest.fixture(scope="module")
def tiny():
    cfg = CONFIGS["tiny"]
    Bp, C, D = make_df_inputs(cfg)
    return cfg, Bp, C, D


def test_brute_force_four_index(tiny):
    cfg, Bp, C, D = tiny
    nao = cfg.nao
    Bf = _full_B(Bp, nao)
    eri = np.einsum("qij,qkl->ijkl", Bf, Bf)  # (ij|kl), PAPER.md:35-43 (Eqs. 1-2)
    J_bf = np.einsum("ijkl,kl->ij", eri, D)
    # K of Eq. 6 has no occupation factor: it equals the exchange contraction
    # with C C^T = D/2 (SURVEY Q7 / reading R8).
    K_bf = np.einsum("ikjl,kl->ij", eri, C @ C.T)
    J, K = O.df_jk_plain(Bp, nao, C, D)
    assert O.rel_frobenius(J, J_bf) < 1e-13
    assert O.rel_frobenius(K, K_bf) < 1e-13
    # and NOT the D = 2CC^T contraction (a factor-2 mistake must fail)
    assert O.rel_frobenius(K, np.einsum("ikjl,kl->ij", eri, D)) > 0.4


def test_invariants(tiny):
    cfg, Bp, C, D = tiny
    nao = cfg.nao
    rho = O.df_rho(Bp, nao, D)
    J, K = O.df_jk_plain(Bp, nao, C, D)
    assert np.array_equal(J, J.T)
    assert np.array_equal(K, K.T)
    # Tr(D J) = |rho|^2
    assert np.trace(D @ J) == pytest.approx(float(rho @ rho), rel=1e-12)
    # K is a Gram matrix: PSD, Tr(D K) = 2 |C^T X|^2 >= 0
    lam = np.linalg.eigvalsh(K)
    assert lam.min() > -1e-10 * lam.max()
    X = O.df_x(Bp, nao, C)
    t = 2.0 * sum(np.linalg.norm(C.T @ X[q]) ** 2 for q in range(cfg.naux))
    assert np.trace(D @ K) == pytest.approx(t, rel=1e-12)
    assert np.trace(D @ K) > 0


def test_rho_uses_both_triangles():
    # D deliberately non-symmetric in storage: only its symmetric part counts
    rng = np.random.default_rng(5)
    nao, naux = 7, 3
    Bp = rng.standard_normal((O.npair(nao), naux))
    Dn = rng.standard_normal((nao, nao))
    Bf = _full_B(Bp, nao)
    Ds = 0.5 * (Dn + Dn.T)
    ref = np.einsum("qij,ij->q", Bf, Ds)
    assert np.allclose(O.df_rho(Bp, nao, Dn), ref, rtol=1e-13, atol=1e-13)


def test_rank_one_case():
    # naux = 1: J = (b . d) b, K = (B C)(B C)^T
    rng = np.random.default_rng(11)
    nao, nocc = 9, 3
    Bp = rng.standard_normal((O.npair(nao), 1))
    C = np.linalg.qr(rng.standard_normal((nao, nao)))[0][:, :nocc]
    D = 2 * C @ C.T
    Bm = _full_B(Bp, nao)[0]
    J, K = O.df_jk_plain(Bp, nao, C, D)
    assert np.allclose(J, np.sum(Bm * D) * Bm, rtol=1e-13, atol=1e-14)
    assert np.allclose(K, (Bm @ C) @ (Bm @ C).T, rtol=1e-13, atol=1e-14)


def test_unpack_matches_pair_index():
    nao = 6
    v = np.arange(O.npair(nao), dtype=np.float64)
    M = O.unpack_sym(v, nao)
    for i in range(nao):
        for j in range(nao):
            assert M[i, j] == v[int(pair_index(i, j))]


def test_flops_model_golden(golden_dir):
    import os

    rows = []
    with open(os.path.join(golden_dir, "flops_paper.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, nao, naux, nocc, jf, kf = line.split()
            rows.append((name, int(nao), int(naux), int(nocc), int(jf), int(kf)))
    assert len(rows) == 4
    for name, nao, naux, nocc, jf, kf in rows:
        cfg = CONFIGS[name]
        assert (cfg.nao, cfg.naux, cfg.nocc) == (nao, naux, nocc)
        fm = O.flops_model(nao, naux, nocc)
        assert fm["J"] == jf and fm["K"] == kf
        # the paper's own formula with N_scr = N_bf^2
        assert fm["K"] == 2 * (nao * nao + nao * nao) * naux * nocc
