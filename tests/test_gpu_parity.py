"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by
element on the same seeded inputs.  Integer work (scale indices, digits, INT32 weight sums) is
bit-exact; the emulated FP64 GEMM follows the oracle's summation order, so it is compared
bit-exactly too (R6) and, separately, within the requested tol against plain FP64."""
import numpy as np
import pytest
import torch

from df_inputs import generators as G
from oracle import df_oracle as O

pytestmark = pytest.mark.gpu
DEV = "cuda"
TOLS = (1e-4, 1e-6, 1e-8, 1e-10)  # BASELINE.json north_star


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).to(DEV)


def assert_k_matches_emulation(K, K_emu):
    """K of the CUDA path against the oracle's emulated K.  X and every GEMM(6) scale index are
    bit-equal, so the two differ only in the order of the FP64 additions over the q-groups (SURVEY.md
    8(c): a tolerance for the last bits): 1e-14 in the Frobenius norm, and no single entry off by more
    than 1e-13 of its Cauchy-Schwarz scale sqrt(K_ii K_jj) -- a norm alone would hide one wrong entry."""
    assert O.rel_frobenius(K, K_emu) <= 1e-14
    d = np.sqrt(np.maximum(np.diag(K_emu), 0.0))
    scale = np.outer(d, d)
    diff = np.abs(K - K_emu)
    assert not diff[scale == 0.0].any()
    assert np.max(diff[scale > 0.0] / scale[scale > 0.0], initial=0.0) <= 1e-13


def edge_matrix(rows, cols, seed):
    """Random wide-range rows plus the scale-index edge cases of DESIGN.md R2."""
    rng = np.random.default_rng(seed)
    X = rng.standard_normal((rows, cols)) * np.exp2(rng.integers(-25, 25, size=(rows, 1)).astype(float))
    X *= np.exp2(rng.uniform(-20, 0, size=(rows, cols)))
    X[0] = 0.0                                   # zero row
    X[1] = 0.0; X[1, cols // 2] = -1.0           # a single power of two
    X[2] *= 1e-3; X[2, 0] = 127.0 / 128.0        # exactly at the bump boundary f = 127/128
    X[3] *= 1e-3; X[3, 1] = np.nextafter(127.0 / 128.0, 0.0)  # just below it
    X[4] *= 1e-3; X[4, 2] = np.nextafter(1.0, 0.0)            # just below a power of two
    X[5] = 2.0 ** -1005                          # below the tiny-row threshold -> zero row
    X[6, :] = np.where(rng.integers(0, 2, cols) > 0, 1.0, -1.0) * 2.0 ** 17  # +-max everywhere
    X[7] = 0.0; X[7, -1] = 3.0e-300              # valid scale, flagged out of range
    return X


@pytest.mark.parametrize("rows,cols", [(37, 1000), (130, 48), (9, 17), (64, 4099)])
@pytest.mark.parametrize("s", [1, 3, 8])
def test_split_rows_bit_exact(dfe, gpu_ws, rows, cols, s):
    X = edge_matrix(max(rows, 8), cols, seed=rows + cols)
    rows = X.shape[0]
    e_ref, D_ref = O.split_operand(X, s)
    pitch = dfe.df_plane_pitch(cols)
    e = torch.empty(rows, dtype=torch.int32, device=DEV)
    pl = torch.full((s, rows, pitch), 99, dtype=torch.int8, device=DEV)
    dfe.df_debug_split_rows(dev(X), rows, cols, s, e, pl)
    torch.cuda.synchronize()
    assert np.array_equal(e.cpu().numpy(), e_ref)
    got = pl.cpu().numpy()
    ok_rows = np.arange(rows) != 7  # row 7 is out of range: flagged, digits unspecified (R9)
    assert np.array_equal(got[:, ok_rows, :cols], D_ref[:, ok_rows])
    assert not got[:, :, cols:].any()  # padding is zero
    assert dfe.df_last_status() == dfe.DF_STATUS_RANGE  # row 7 only
    assert O.operand_status(X) == 2


@pytest.mark.parametrize("k,n", [(1000, 37), (48, 130), (33, 9), (300, 1000)])
@pytest.mark.parametrize("s", [2, 5, 8])
def test_split_cols_bit_exact(dfe, gpu_ws, k, n, s):
    Xt = edge_matrix(max(n, 8), k, seed=k * 3 + n)  # rows = columns of the k x n operand
    n = Xt.shape[0]
    X = np.ascontiguousarray(Xt.T)
    e_ref, D_ref = O.split_operand(Xt, s)
    pitch = dfe.df_plane_pitch(k)
    e = torch.empty(n, dtype=torch.int32, device=DEV)
    pl = torch.full((s, n, pitch), 99, dtype=torch.int8, device=DEV)
    dfe.df_debug_split_cols(dev(X), k, n, s, e, pl)
    torch.cuda.synchronize()
    assert np.array_equal(e.cpu().numpy(), e_ref)
    got = pl.cpu().numpy()
    ok_cols = np.arange(n) != 7  # column 7 is out of range: flagged, digits unspecified (R9)
    assert np.array_equal(got[:, ok_cols, :k], D_ref[:, ok_cols])
    assert not got[:, :, k:].any()
    assert dfe.df_last_status() == dfe.DF_STATUS_RANGE


def test_status_word_flags_nonfinite(dfe, gpu_ws):
    X = np.ones((4, 64)); X[2, 5] = np.inf
    e = torch.empty(4, dtype=torch.int32, device=DEV)
    pl = torch.empty((2, 4, 64), dtype=torch.int8, device=DEV)
    dfe.df_last_status()
    dfe.df_debug_split_rows(dev(X), 4, 64, 2, e, pl)
    assert dfe.df_last_status() & dfe.DF_STATUS_NONFINITE
    assert dfe.df_last_status() == 0  # cleared by the read
    assert O.operand_status(X) & 1


def random_digits(s, rows, k, seed):
    rng = np.random.default_rng(seed)
    pitch = (k + 31) // 32 * 32
    D = np.full((s, rows, pitch), 77, dtype=np.int8)  # garbage past k must never be read
    D[:, :, :k] = rng.integers(-128, 128, size=(s, rows, k))
    D[:, 0, :k] = -128  # extreme rows: the INT32 guard's worst case
    D[:, -1, :k] = 127
    return D


@pytest.mark.parametrize("bk", [32, 64, 128])
@pytest.mark.parametrize("m,n,k,s", [
    (128, 128, 128, 1),     # one tile, one slice pair: P^(1,1)
    (300, 200, 1000, 4),    # several tiles, ragged tails in m, n, k
    (130, 160, 1200, 3),    # GEMM(5)-like: n_tile = 160 -> 3 weights per pass, 1 pass
    (257, 48, 777, 5),      # narrow N, all 5 weights in TMEM
    (129, 250, 96, 8),      # two N tiles, two passes of 4 weights
])
def test_weight_sums_int32_bit_exact(dfe, gpu_ws, bk, m, n, k, s):
    DA, DB = random_digits(s, m, k, 11), random_digits(s, n, k, 12)
    P = torch.full((s, m, n), -12345, dtype=torch.int32, device=DEV)
    dfe.df_debug_weight_sums(dev(DA), dev(DB), m, n, k, s, 0, bk, P)
    torch.cuda.synchronize()
    ref = O.weight_sums(DA[:, :, :k], DB[:, :, :k], s)
    got = P.cpu().numpy()
    for w in range(2, s + 2):
        assert np.array_equal(got[w - 2], ref[w]), f"w={w}"


@pytest.mark.parametrize("s,k", [(8, 16352 + 2000), (3, 43680 + 64)])
def test_weight_sums_flush_chunks(dfe, gpu_ws, s, k):
    """k > kflush(s): every chunk's INT32 sums are exact and the worst case does not overflow."""
    m, n = 128, 64
    DA, DB = random_digits(s, m, k, 21), random_digits(s, n, k, 22)
    kf = dfe.df_kflush(s)
    P = torch.empty((s, m, n), dtype=torch.int32, device=DEV)
    for ch in range((k + kf - 1) // kf):
        dfe.df_debug_weight_sums(dev(DA), dev(DB), m, n, k, s, ch, 0, P)
        torch.cuda.synchronize()
        ref = O.weight_sums(DA[:, :, :k], DB[:, :, :k], s, ch * kf, min(k, (ch + 1) * kf))
        got = P.cpu().numpy()
        for w in range(2, s + 2):
            assert np.abs(ref[w]).max() < 2 ** 31
            assert np.array_equal(got[w - 2], ref[w]), f"chunk {ch} w={w}"


# n % 4 == 0: 256-bit epilogue accesses; n = 250: 16-byte staged path; odd n: scalar path
@pytest.mark.parametrize("m,n,k", [(256, 256, 256), (300, 200, 1000), (128, 48, 4096), (1, 1, 1), (5, 700, 33),
                                   (200, 250, 520), (37, 131, 200)])
def test_emul_gemm_matches_oracle_emulation_bitwise(dfe, gpu_ws, m, n, k):
    A, B = G.make_gemm_inputs(m, n, k, seed=3)
    Ad, Bd = dev(A), dev(B)
    for s in range(1, 9):
        C = torch.empty((m, n), dtype=torch.float64, device=DEV)
        dfe.df_emul_gemm_slices(Ad, Bd, C, m, n, k, s)
        torch.cuda.synchronize()
        assert np.array_equal(C.cpu().numpy(), O.emul_gemm(A, B, s)), f"s={s}"
    assert dfe.df_last_status() == 0


def test_emul_gemm_two_flush_chunks_bitwise(dfe, gpu_ws):
    m, n, k, s = 130, 70, 16352 + 1500, 8
    A, B = G.make_gemm_inputs(m, n, k, seed=8)
    C = torch.empty((m, n), dtype=torch.float64, device=DEV)
    dfe.df_emul_gemm_slices(dev(A), dev(B), C, m, n, k, s)
    torch.cuda.synchronize()
    assert np.array_equal(C.cpu().numpy(), O.emul_gemm(A, B, s))


@pytest.mark.parametrize("tol", TOLS)
def test_emul_gemm_within_tol(dfe, gpu_ws, tol):
    m, n, k = 512, 384, 2048
    A, B = G.make_gemm_inputs(m, n, k, seed=4)
    C = torch.empty((m, n), dtype=torch.float64, device=DEV)
    dfe.df_emul_gemm(dev(A), dev(B), C, m, n, k, tol)
    torch.cuda.synchronize()
    err = O.rel_frobenius(C.cpu().numpy(), O.gemm_plain(A, B))
    assert err <= tol, (err, tol, dfe.df_slices_for_tol(tol))


def test_emul_gemm_max_slices_1e12(dfe, gpu_ws):
    m, n, k = 256, 256, 1024
    A, B = G.make_gemm_inputs(m, n, k, seed=5)
    C = torch.empty((m, n), dtype=torch.float64, device=DEV)
    dfe.df_emul_gemm_slices(dev(A), dev(B), C, m, n, k, 8)
    torch.cuda.synchronize()
    ref = O.gemm_longdouble(A, B)
    err = float(np.linalg.norm((C.cpu().numpy() - ref).astype(np.float64)) / np.linalg.norm(ref.astype(np.float64)))
    assert err <= 1e-12, err


def test_emul_gemm_zero_and_degenerate(dfe, gpu_ws):
    A = np.zeros((40, 50)); B = np.random.default_rng(0).standard_normal((50, 30))
    C = torch.full((40, 30), 7.0, dtype=torch.float64, device=DEV)
    dfe.df_emul_gemm_slices(dev(A), dev(B), C, 40, 30, 50, 4)
    torch.cuda.synchronize()
    assert not C.cpu().numpy().any()
    with pytest.raises(dfe.DFError):
        dfe.df_emul_gemm_slices(dev(A), dev(B), C, 0, 30, 50, 4)  # empty input is an argument error


def run_jk(dfe, Bp, cfg_nao, naux, Cocc, nocc, D, s, want_x=True):
    a_pad = (nocc + 15) // 16 * 16
    J = torch.empty((cfg_nao, cfg_nao), dtype=torch.float64, device=DEV)
    K = torch.empty_like(J)
    X = torch.zeros((naux, cfg_nao, a_pad), dtype=torch.float64, device=DEV) if want_x else None
    e6 = torch.zeros((4096, cfg_nao), dtype=torch.int32, device=DEV)
    ng = dfe.df_debug_jk_build(dev(Bp), cfg_nao, naux, dev(Cocc), nocc, dev(D), s, J, K, X, e6)
    torch.cuda.synchronize()
    return J.cpu().numpy(), K.cpu().numpy(), (X.cpu().numpy() if want_x else None), e6.cpu().numpy()[:ng], ng


@pytest.mark.parametrize("tol", [1e-4, 1e-8, 1e-12])
def test_jk_tiny_config0(dfe, gpu_ws, tol):
    cfg = G.CONFIGS["tiny"]
    Bp, Cocc, D = G.make_df_inputs(cfg)
    s = dfe.df_slices_for_tol(tol)
    J, K, X, e6, ng = run_jk(dfe, Bp, cfg.nao, cfg.naux, Cocc, cfg.nocc, D, s)
    J_ref, K_ref = O.df_jk_plain(Bp, cfg.nao, Cocc, D)
    K_emu, X_emu = O.emul_df_k(Bp, cfg.nao, Cocc, s, return_x=True)
    assert O.rel_frobenius(J, J_ref) <= 1e-12
    assert O.rel_frobenius(K, K_ref) <= tol
    # stage by stage: GEMM(5) output bit-exact, GEMM(6) scales exact, K up to FP64 summation order
    assert np.array_equal(X[:, :, :cfg.nocc], X_emu)
    assert not X[:, :, cfg.nocc:].any()
    groups = O.q_groups(cfg.naux, cfg.nocc, s)
    assert ng == len(groups)
    for g, (g0, g1) in enumerate(groups):
        Xrow = np.transpose(X_emu[g0:g1], (1, 0, 2)).reshape(cfg.nao, -1)
        assert np.array_equal(e6[g], O.scale_index(np.max(np.abs(Xrow), axis=1)))
    assert_k_matches_emulation(K, K_emu)
    assert np.array_equal(J, J.T) and np.array_equal(K, K.T)
    assert np.linalg.eigvalsh(K).min() >= -1e-12 * np.abs(K).max()
    assert dfe.df_last_status() == 0
    # the same call through the tol entry point gives the same bits
    J2 = torch.empty((cfg.nao, cfg.nao), dtype=torch.float64, device=DEV); K2 = torch.empty_like(J2)
    dfe.df_jk_build(dev(Bp), cfg.nao, cfg.naux, dev(Cocc), cfg.nocc, dev(D), tol, J2, K2)
    torch.cuda.synchronize()
    assert np.array_equal(K2.cpu().numpy(), K)


def test_jk_many_groups_and_superblocks(dfe, gpu_ws):
    """naux spans three 512-blocks (ragged last one), two q-groups per full block, ragged nao/nocc;
    a minimum-size workspace forces one super-block per 512 q and must give the same bits."""
    nao, naux, nocc, s = 40, 1100, 40, 8
    Bp = G.make_B_packed(nao, naux, seed=7)
    Cocc = G.make_C_occ(nao, nocc, seed=7)
    D = G.make_density(Cocc)
    groups = O.q_groups(naux, nocc, s)
    assert len(groups) == 5  # 408 + 104 | 408 + 104 | 76
    J, K, X, e6, ng = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
    K_emu, X_emu = O.emul_df_k(Bp, nao, Cocc, s, return_x=True)
    J_ref, K_ref = O.df_jk_plain(Bp, nao, Cocc, D)
    assert ng == 5
    assert np.array_equal(X[:, :, :nocc], X_emu)
    for g, (g0, g1) in enumerate(groups):
        Xrow = np.transpose(X_emu[g0:g1], (1, 0, 2)).reshape(nao, -1)
        assert np.array_equal(e6[g], O.scale_index(np.max(np.abs(Xrow), axis=1)))
    assert_k_matches_emulation(K, K_emu)
    assert O.rel_frobenius(K, K_ref) <= 1e-12 and O.rel_frobenius(J, J_ref) <= 1e-12
    small = dfe.Workspace(dfe.df_jk_workspace_bytes(nao, naux, nocc, s))
    try:
        J2, K2, X2, e62, ng2 = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
    finally:
        small.close()
        dfe.df_set_workspace(gpu_ws.view)
    assert ng2 == 5 and np.array_equal(K2, K) and np.array_equal(X2, X) and np.array_equal(J2, J)


@pytest.mark.parametrize("nocc,s,naux", [(70, 4, 1000), (141, 3, 700), (45, 8, 1030), (65, 5, 600), (105, 6, 530)])
def test_jk_group_boundaries_off_32(dfe, gpu_ws, nocc, s, naux):
    """q-groups whose padded width |g| pad16(nocc) is NOT a multiple of 32 bytes (the K extent of one
    MMA): a_pad = 16 * odd and an odd group length.  planes6 starts every group on a multiple of 32
    columns with zero bytes in between, so no MMA of GEMM(6) reads digits of the next group
    (they were made with another scale).  X bit-exact, e6 exact, K against the oracle's emulation."""
    nao = 40
    a_pad = (nocc + 15) // 16 * 16
    groups = O.q_groups(naux, nocc, s)
    assert len(groups) >= 2 and a_pad % 32 == 16
    assert any(((g1 - g0) * a_pad) % 32 == 16 for g0, g1 in groups[:-1])
    Bp = G.make_B_packed(nao, naux, seed=50 + s)
    Cocc = G.make_C_occ(max(nao, nocc), nocc, seed=50 + s)[:nao]  # nocc may exceed nao: any nao x nocc matrix
    D = G.make_density(Cocc)
    J, K, X, e6, ng = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
    K_emu, X_emu = O.emul_df_k(Bp, nao, Cocc, s, return_x=True)
    assert ng == len(groups)
    assert np.array_equal(X[:, :, :nocc], X_emu)
    for g, (g0, g1) in enumerate(groups):
        Xrow = np.transpose(X_emu[g0:g1], (1, 0, 2)).reshape(nao, -1)
        assert np.array_equal(e6[g], O.scale_index(np.max(np.abs(Xrow), axis=1)))
    assert_k_matches_emulation(K, K_emu)
    assert np.array_equal(K, K.T) and dfe.df_last_status() == 0


@pytest.mark.parametrize("s", [4, 5, 6, 8])
def test_jk_split_n_tiles(dfe, gpu_ws, s):
    """nocc = 150 (config 3's value): a_pad = 160 does not fit s accumulators in TMEM.  s = 4: the
    whole a_pad on MMA pairs in two passes; s = 5, 6: two N halves of 80 columns, one pass each, as
    256-row tiles on MMA pairs; s = 8: the halves on multicast CTA pairs in two passes with the FP64
    read-modify-write.  Ragged nao, several M tiles straddling q boundaries."""
    nao, naux, nocc = 168, 38 if s == 4 else 37, 150  # even naux: fused GEMM(5); odd: separate unpack
    Bp = G.make_B_packed(nao, naux, seed=13)
    Cocc = G.make_C_occ(nao, nocc, seed=13)
    D = G.make_density(Cocc)
    J, K, X, e6, ng = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
    K_emu, X_emu = O.emul_df_k(Bp, nao, Cocc, s, return_x=True)
    J_ref, K_ref = O.df_jk_plain(Bp, nao, Cocc, D)
    assert np.array_equal(X[:, :, :nocc], X_emu)
    assert not X[:, :, nocc:].any()
    assert_k_matches_emulation(K, K_emu)
    assert O.rel_frobenius(J, J_ref) <= 1e-12
    assert O.rel_frobenius(K, K_ref) <= {4: 1e-6, 5: 1e-9, 6: 1e-11, 8: 1e-12}[s]  # 2^(8 - 8 s) and margin
    assert dfe.df_last_status() == 0


@pytest.mark.parametrize("s", [1, 2, 3, 4, 5, 6, 7, 8])
def test_jk_every_slice_count_ragged(dfe, gpu_ws, s):
    """Every template instantiation of the unpack / split kernels (s = 1..8) on a ragged case:
    nao = 137 (one full 128-tile + 9 rows, last 16-column group partial), naux = 77 (two full
    32-q chunks + 13), nocc = 21 (a_pad 32).  GEMM(5) output bit-exact, K up to summation order."""
    nao, naux, nocc = 137, 77, 21
    Bp = G.make_B_packed(nao, naux, seed=40 + s)
    Cocc = G.make_C_occ(nao, nocc, seed=40 + s)
    D = G.make_density(Cocc)
    J, K, X, e6, ng = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
    K_emu, X_emu = O.emul_df_k(Bp, nao, Cocc, s, return_x=True)
    J_ref, _ = O.df_jk_plain(Bp, nao, Cocc, D)
    assert np.array_equal(X[:, :, :nocc], X_emu)
    assert not X[:, :, nocc:].any()
    assert_k_matches_emulation(K, K_emu)
    assert O.rel_frobenius(J, J_ref) <= 1e-12
    assert np.array_equal(K, K.T) and dfe.df_last_status() == 0


@pytest.mark.parametrize("smax", [4, 8])
def test_jk_planned_build_bitwise(dfe, gpu_ws, smax):
    """B split once (row maxima, scale indices, smax digit planes)
    and reused; a planned build with s <= smax slices reads the first s planes (prefix property,
    DESIGN.md R3) and must give the bits of df_jk_build -- which the other tests compare with the
    oracle -- for several (C_occ, D) of an SCF-like sequence, ragged nao, 3 blocks of 512 q."""
    nao, naux, nocc = 150, 1100, 20
    Bp = G.make_B_packed(nao, naux, seed=21)
    Bd = dev(Bp)
    plan = dfe.Plan(Bd, nao, naux, smax)
    assert dfe.df_last_status() == 0
    for it, s in enumerate([2, 3, 4] if smax == 4 else [4, 6, 8]):
        Cocc = G.make_C_occ(nao, nocc, seed=30 + it)
        D = G.make_density(Cocc)
        J = torch.empty((nao, nao), dtype=torch.float64, device=DEV)
        K = torch.empty_like(J)
        dfe.df_jk_build_slices(Bd, nao, naux, dev(Cocc), nocc, dev(D), s, J, K)
        J2 = torch.full_like(J, np.nan)
        K2 = torch.full_like(K, np.nan)
        dfe.df_jk_build_planned_slices(plan, Bd, nao, naux, dev(Cocc), nocc, dev(D), s, J2, K2)
        torch.cuda.synchronize()
        assert torch.equal(J, J2) and torch.equal(K, K2), s
        K_emu = O.emul_df_k(Bp, nao, Cocc, s)
        assert_k_matches_emulation(K2.cpu().numpy(), K_emu)
    # tol entry point: same policy as df_jk_build
    tol = 1e-6
    dfe.df_jk_build(Bd, nao, naux, dev(Cocc), nocc, dev(D), tol, J, K)
    if dfe.df_slices_for_tol(tol) <= smax:
        dfe.df_jk_build_planned(plan, Bd, nao, naux, dev(Cocc), nocc, dev(D), tol, J2, K2)
        torch.cuda.synchronize()
        assert torch.equal(J, J2) and torch.equal(K, K2)
    assert dfe.df_last_status() == 0
    # more slices than the plan holds, a plan buffer that is too small
    with pytest.raises(dfe.DFError) as ei:
        dfe.df_jk_build_planned_slices(plan, Bd, nao, naux, dev(Cocc), nocc, dev(D), smax + 1 if smax < 8 else 9, J2, K2)
    assert ei.value.code == -3
    small = torch.empty(dfe.df_jk_plan_bytes(nao, naux, smax) - 1 + 256, dtype=torch.uint8, device=DEV)
    off = (-small.data_ptr()) % 256
    rc = dfe.lib.df_jk_plan_create(Bd.data_ptr(), nao, naux, smax, small.data_ptr() + off,
                                   dfe.df_jk_plan_bytes(nao, naux, smax) - 1, None)
    assert rc == -4
    plan.close()


def test_jk_planned_small_workspace(dfe, gpu_ws):
    """A planned build in the planned workspace of one 512-q block (no GEMM(5) planes in it)."""
    nao, naux, nocc, s = 150, 1100, 20, 5
    Bp = G.make_B_packed(nao, naux, seed=22)
    Cocc = G.make_C_occ(nao, nocc, seed=22)
    D = G.make_density(Cocc)
    Bd = dev(Bp)
    J = torch.empty((nao, nao), dtype=torch.float64, device=DEV)
    K = torch.empty_like(J)
    dfe.df_jk_build_slices(Bd, nao, naux, dev(Cocc), nocc, dev(D), s, J, K)
    plan = dfe.Plan(Bd, nao, naux, 6)
    small = dfe.Workspace(dfe.df_jk_planned_workspace_bytes(nao, naux, nocc, s, 1))
    try:
        assert small.view.numel() < dfe.df_jk_workspace_bytes(nao, naux, nocc, s)
        J2, K2 = torch.empty_like(J), torch.empty_like(K)
        dfe.df_jk_build_planned_slices(plan, Bd, nao, naux, dev(Cocc), nocc, dev(D), s, J2, K2)
        torch.cuda.synchronize()
        with pytest.raises(dfe.DFError) as ei:  # the unplanned build does not fit there
            dfe.df_jk_build_slices(Bd, nao, naux, dev(Cocc), nocc, dev(D), s, J2.clone(), K2.clone())
        assert ei.value.code == -4
    finally:
        small.close()
        dfe.df_set_workspace(gpu_ws.view)
    assert torch.equal(J, J2) and torch.equal(K, K2)


def test_jk_workspace_too_small(dfe, gpu_ws):
    tiny = dfe.Workspace(4096)
    try:
        with pytest.raises(dfe.DFError) as ei:
            run_jk(dfe, *G.make_df_inputs(G.CONFIGS["tiny"])[:1], 48, 160, np.zeros((48, 10)), 10, np.zeros((48, 48)), 3)
        assert ei.value.code == -4
    finally:
        tiny.close()
        dfe.df_set_workspace(gpu_ws.view)


def test_jk_naux_1_rank_one(dfe, gpu_ws):
    """naux = 1: J = (b.d) b and K = (B C)(B C)^T, the textbook special case."""
    nao, nocc = 33, 7
    Bp = G.make_B_packed(nao, 1, seed=9)
    Cocc = G.make_C_occ(nao, nocc, seed=9)
    D = G.make_density(Cocc)
    J, K, _, _, ng = run_jk(dfe, Bp, nao, 1, Cocc, nocc, D, 8)
    Bm = O.unpack_sym(Bp[:, 0], nao)
    assert ng == 1
    assert np.allclose(J, np.sum(Bm * D) * Bm, rtol=1e-12, atol=1e-14 * np.abs(Bm).max())
    assert O.rel_frobenius(K, (Bm @ Cocc) @ (Bm @ Cocc).T) <= 1e-12


def test_jk_medium_config2(dfe, gpu_ws):
    """BASELINE.json config 2 (nao 500, naux 1700, nocc 50): several M tiles per q, four 512-q blocks,
    full plain-FP64 oracle for J and K, oracle emulation for sampled q (bit-exact X)."""
    cfg = G.CONFIGS["medium"]
    Bp, Cocc, D = G.make_df_inputs(cfg)
    J_ref, K_ref = O.df_jk_plain(Bp, cfg.nao, Cocc, D)
    for tol in (1e-6, 1e-10):
        s = dfe.df_slices_for_tol(tol)
        J, K, X, e6, ng = run_jk(dfe, Bp, cfg.nao, cfg.naux, Cocc, cfg.nocc, D, s)
        assert ng == len(O.q_groups(cfg.naux, cfg.nocc, s))
        assert O.rel_frobenius(J, J_ref) <= 1e-12
        assert O.rel_frobenius(K, K_ref) <= tol
        assert np.array_equal(K, K.T) and np.array_equal(J, J.T)
        for q in (0, 511, 512, 1699):
            Xq = O.emul_x_group(Bp, cfg.nao, Cocc, s, q, q + 1)[0]
            assert np.array_equal(X[q, :, :cfg.nocc], Xq), f"q={q}"
    assert dfe.df_last_status() == 0


_CONFIG4_REF = {}  # the oracle's J (all q) and K (first 512 q) of config 4, computed once per session


def config4_oracle_refs(B, cfg, Cocc, D, qs):
    """The oracle's plain FP64 J over all of config 4 (rho_q and J are sums over q, Eqs. 3-4: the 78 GB
    of device bytes are streamed to the host in 512-q blocks, about a minute) and its K over the first
    `qs` auxiliary functions (Eq. 6; K over all 6000 would take ten minutes)."""
    if not _CONFIG4_REF:
        nao, naux = cfg.nao, cfg.naux
        rho = np.empty(naux)
        J_ref = np.zeros((nao, nao))
        K_ref = None
        for q0 in range(0, naux, 512):
            q1 = min(naux, q0 + 512)
            Bb = B[:, q0:q1].contiguous().cpu().numpy()
            rho[q0:q1] = O.df_rho(Bb, nao, D)
            J_ref += O.df_j(Bb, nao, rho[q0:q1])
            if q0 == 0:
                K_ref = O.df_k(Bb[:, :qs], nao, Cocc)
            del Bb
        _CONFIG4_REF.update(J_ref=J_ref, K_ref=K_ref, rho=rho)
    return _CONFIG4_REF


@pytest.mark.parametrize("tol", [1e-6, 1e-10])
def test_jk_largest_config4(dfe, gpu_ws, tol):
    """BASELINE.json config 4 at full size (nao 1800, naux 6000, nocc 250; packed B 78 GB on the
    device, naux processed in super-blocks of two 512-q blocks) at both tolerances it names
    (s = 4: GEMM(5) as two 128-column N tiles on MMA pairs; s = 6: on multicast CTA pairs with a
    second pass).  X of sampled q bit for bit against the oracle's emulation of GEMM(5) from the same
    bytes, every GEMM(6) scale index exactly, J as a FULL matrix against the oracle's plain FP64 J of the
    same bytes (<= 1e-12), K as a full matrix on a 512-q sub-build (the shape of bench.py's parity
    check) against the oracle's K within tol, norm and element-wise, sampled entries of the full-size K
    against the oracle's definition, symmetry and the trace invariants.  (The oracle's K over all 6000 q
    of this size takes ~10 minutes of host time: the full-size full-matrix K comparison is the config-3 test.)"""
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 140 << 30:
        pytest.skip("needs ~135 GB of free device memory")
    cfg = G.CONFIGS["largest"]
    nao, naux, nocc = cfg.nao, cfg.naux, cfg.nocc
    a_pad = (nocc + 15) // 16 * 16
    s = dfe.df_slices_for_tol(tol)
    assert s == (4 if tol == 1e-6 else 6)  # guarded policy (R7): ceil((log2(1/tol) + 7) / 8)
    B = G.make_B_packed_torch(nao, naux, cfg.seed, device=DEV)
    Cocc = G.make_C_occ(nao, nocc, cfg.seed)
    D = G.make_density(Cocc)
    big = dfe.Workspace(dfe.df_jk_workspace_bytes_blocks(nao, naux, nocc, s, 2))  # 1024 q per launch
    try:
        J = torch.empty((nao, nao), dtype=torch.float64, device=DEV)
        K = torch.empty_like(J)
        dfe.df_jk_build(B, nao, naux, dev(Cocc), nocc, dev(D), tol, J, K)
        torch.cuda.synchronize()
        assert dfe.df_last_status() == 0
        J2, K2 = torch.full_like(J, np.nan), torch.full_like(K, np.nan)
        X = torch.empty((naux, nao, a_pad), dtype=torch.float64, device=DEV)
        e6 = torch.zeros((256, nao), dtype=torch.int32, device=DEV)
        ng = dfe.df_debug_jk_build(B, nao, naux, dev(Cocc), nocc, dev(D), s, J2, K2, X, e6)
        torch.cuda.synchronize()
        assert torch.equal(J, J2) and torch.equal(K, K2)
        groups = O.q_groups(naux, nocc, s)
        assert ng == len(groups)
        eC, DC = O.split_operand(np.ascontiguousarray(Cocc.T), s)
        for q in (0, 1023, 1024, groups[7][0], 5631, 5999):  # super-block, block and group boundaries, the ragged tail
            Bq = B[:, q:q + 1].contiguous().cpu().numpy()
            Xq = O.emul_x_group(Bq, nao, Cocc, s, 0, 1, eC, DC)[0]
            got = X[q].cpu().numpy()
            assert np.array_equal(got[:, :nocc], Xq), f"q={q}"
            assert not got[:, nocc:].any()
        e6h = e6.cpu().numpy()
        for g, (g0, g1) in enumerate(groups):
            m = X[g0:g1].abs().amax(dim=(0, 2)).cpu().numpy()
            assert np.array_equal(e6h[g], O.scale_index(m)), f"group {g}"
        del X, J2, K2
        # the first 512 q as a build of their own: K as a full matrix against the oracle
        qs = 512
        ref = config4_oracle_refs(B, cfg, Cocc, D, qs)
        Bs = B[:, :qs].contiguous()
        Js, Ks = torch.empty_like(J), torch.empty_like(K)
        dfe.df_jk_build(Bs, nao, qs, dev(Cocc), nocc, dev(D), tol, Js, Ks)
        torch.cuda.synchronize()
        Ksh = Ks.cpu().numpy()
        del Bs, Js, Ks
        eKs = O.rel_frobenius(Ksh, ref["K_ref"])
        assert eKs <= tol, (eKs, tol, s)
        dK = np.sqrt(np.diag(ref["K_ref"]))
        assert np.max(np.abs(Ksh - ref["K_ref"]) / np.outer(dK, dK)) <= tol
    finally:
        big.close()
        dfe.df_set_workspace(gpu_ws.view)
    Jh, Kh = J.cpu().numpy(), K.cpu().numpy()
    assert np.array_equal(Jh, Jh.T) and np.array_equal(Kh, Kh.T)
    assert np.isfinite(Jh).all() and np.isfinite(Kh).all()
    # J over all 6000 q, full matrix (J is plain FP64 on both sides: PAPER.md:101)
    eJ = O.rel_frobenius(Jh, ref["J_ref"])
    assert eJ <= 1e-12, eJ
    rho = ref["rho"]
    assert abs(np.sum(D * Jh) - rho @ rho) <= 1e-11 * (rho @ rho)  # Tr(D J) = |rho|^2

    def x_rows(i):  # X_i[q, a] = sum_j B^q_ij C_ja from the packed rows of i (Eq. 5)
        idx = torch.tensor([max(i, j) * (max(i, j) + 1) // 2 + min(i, j) for j in range(nao)], device=DEV)
        return B.index_select(0, idx).cpu().numpy().T @ Cocc  # (naux, nocc)
    rows = {i: x_rows(i) for i in (0, 911, 1799)}
    for i in rows:
        for j in rows:
            kij = float(np.sum(rows[i] * rows[j]))  # Eq. 6
            scale = np.sqrt(np.sum(rows[i] ** 2) * np.sum(rows[j] ** 2))
            assert abs(Kh[i, j] - kij) <= tol * scale, (i, j, Kh[i, j], kij)
    assert np.sum(D * Kh) >= 0.0
    del B


@pytest.fixture(scope="module")
def config3(dfe):
    """Config 3 (nao 1200, naux 4000, nocc 150; packed B 23 GB generated on the device) and the
    oracle's plain FP64 J and K of it, computed ONCE per session from the same device bytes streamed
    to the host in 512-q blocks (rho_q, J and K are sums over q: Eqs. 3, 4, 6 -- about two minutes of
    host time)."""
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 100 << 30:
        pytest.skip("needs ~90 GB of free device memory")
    cfg = G.CONFIGS["large"]
    nao, naux, nocc = cfg.nao, cfg.naux, cfg.nocc
    B = G.make_B_packed_torch(nao, naux, cfg.seed, device=DEV)
    Cocc = G.make_C_occ(nao, nocc, cfg.seed)
    D = G.make_density(Cocc)
    J_ref = np.zeros((nao, nao))
    K_ref = np.zeros((nao, nao))
    rho = np.empty(naux)
    for q0 in range(0, naux, 512):
        q1 = min(naux, q0 + 512)
        Bb = B[:, q0:q1].contiguous().cpu().numpy()
        rho[q0:q1] = O.df_rho(Bb, nao, D)
        J_ref += O.df_j(Bb, nao, rho[q0:q1])
        K_ref += O.df_k(Bb, nao, Cocc)
        del Bb
    return {"cfg": cfg, "B": B, "Cocc": Cocc, "D": D, "J_ref": J_ref, "K_ref": K_ref, "rho": rho}


# measured rel-F error of the K path with s slices on the configs' data is 2-6e-9 / 5-9e-12 / 3-10e-14
# at s = 4 / 5 / 6; the bound below is the requested tol itself
@pytest.mark.parametrize("tol", [2.0 ** -23, 2.0 ** -31, 2.0 ** -39])
def test_jk_large_config3(dfe, gpu_ws, config3, tol):
    """The benchmark's own launches (bench.py: config 3, all 4000 q in one super-block, the three
    tolerances of the 12-step schedule = Table 1 levels 4, 3, 2, PAPER.md:141-147 -> s = 4, 5, 6 in
    guarded mode) against the oracle: X of sampled q bit for bit (first / last q of 512-blocks, group
    boundaries, the ragged last block), every GEMM(6) scale index exactly, J and K as FULL matrices
    against the oracle's plain FP64 result of the same bytes within 1e-12 / tol, run-to-run and
    plain-vs-planned bit equality."""
    cfg, B, Cocc, D = config3["cfg"], config3["B"], config3["Cocc"], config3["D"]
    nao, naux, nocc = cfg.nao, cfg.naux, cfg.nocc
    a_pad = (nocc + 15) // 16 * 16
    s = dfe.df_slices_for_tol(tol)
    assert s == {2.0 ** -23: 4, 2.0 ** -31: 5, 2.0 ** -39: 6}[tol]
    big = dfe.Workspace(dfe.df_jk_workspace_bytes_blocks(nao, naux, nocc, s, 8))
    try:
        J = torch.empty((nao, nao), dtype=torch.float64, device=DEV)
        K = torch.empty_like(J)
        dfe.df_jk_build(B, nao, naux, dev(Cocc), nocc, dev(D), tol, J, K)
        torch.cuda.synchronize()
        assert dfe.df_last_status() == 0
        # the same build with X and the GEMM(6) scales exported: same bits, every reduction has a fixed order
        J2, K2 = torch.full_like(J, np.nan), torch.full_like(K, np.nan)
        X = torch.empty((naux, nao, a_pad), dtype=torch.float64, device=DEV)
        e6 = torch.zeros((256, nao), dtype=torch.int32, device=DEV)
        ng = dfe.df_debug_jk_build(B, nao, naux, dev(Cocc), nocc, dev(D), s, J2, K2, X, e6)
        torch.cuda.synchronize()
        assert torch.equal(J, J2) and torch.equal(K, K2)
        groups = O.q_groups(naux, nocc, s)
        assert ng == len(groups)
        # X of sampled q, bit for bit (the oracle emulates GEMM(5) for that q from the same bytes)
        gb = [g0 for g0, _ in groups]
        qs = sorted({0, 1, 511, 512, gb[1] - 1, gb[1], 2047, 2048, gb[len(gb) // 2], 3583, 3584, 3999})
        eC, DC = O.split_operand(np.ascontiguousarray(Cocc.T), s)
        for q in qs:
            Bq = B[:, q:q + 1].contiguous().cpu().numpy()
            Xq = O.emul_x_group(Bq, nao, Cocc, s, 0, 1, eC, DC)[0]
            got = X[q].cpu().numpy()
            assert np.array_equal(got[:, :nocc], Xq), f"q={q}"
            assert not got[:, nocc:].any()
        # every scale index of GEMM(6): the oracle's step 1 on the maxima of the exported X per (i, group)
        e6h = e6.cpu().numpy()
        for g, (g0, g1) in enumerate(groups):
            m = X[g0:g1].abs().amax(dim=(0, 2)).cpu().numpy()
            assert np.array_equal(e6h[g], O.scale_index(m)), f"group {g}"
        del X
        # a planned build (B split once) gives the same bits
        plan = dfe.Plan(B, nao, naux, s)
        J2.fill_(np.nan); K2.fill_(np.nan)
        dfe.df_jk_build_planned(plan, B, nao, naux, dev(Cocc), nocc, dev(D), tol, J2, K2)
        torch.cuda.synchronize()
        assert dfe.df_last_status() == 0
        assert torch.equal(J, J2) and torch.equal(K, K2)
        plan.close()
        del J2, K2, plan
    finally:
        big.close()
        dfe.df_set_workspace(gpu_ws.view)
    Jh, Kh = J.cpu().numpy(), K.cpu().numpy()
    assert np.array_equal(Jh, Jh.T) and np.array_equal(Kh, Kh.T)
    eJ = O.rel_frobenius(Jh, config3["J_ref"])
    eK = O.rel_frobenius(Kh, config3["K_ref"])
    assert eJ <= 1e-12, eJ
    assert eK <= tol, (eK, tol, s)
    # element-wise as well: no entry is off by more than tol relative to the Cauchy-Schwarz scale of K
    dK = np.sqrt(np.diag(config3["K_ref"]))
    assert np.max(np.abs(Kh - config3["K_ref"]) / np.outer(dK, dK)) <= tol
    rho = config3["rho"]
    assert abs(np.sum(D * Jh) - rho @ rho) <= 1e-11 * (rho @ rho)  # Tr(D J) = |rho|^2
    assert np.sum(D * Kh) >= 0.0  # Tr(D K) = 2 |C^T X|^2 (R8)


@pytest.mark.parametrize("s", [4, 6])
def test_jk_nocc_250_like(dfe, gpu_ws, s):
    """nocc = 250 (config 4's value): a_pad = 256, GEMM(5) runs two N tiles of 128 columns: on MMA
    pairs in one pass at s = 4, on multicast CTA pairs at s = 6 (a second pass with the running sum
    parked in TMEM)."""
    nao, naux, nocc = 264, 12, 250
    Bp = G.make_B_packed(nao, naux, seed=17)
    Cocc = G.make_C_occ(nao, nocc, seed=17)
    D = G.make_density(Cocc)
    J, K, X, e6, ng = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
    K_emu, X_emu = O.emul_df_k(Bp, nao, Cocc, s, return_x=True)
    J_ref, K_ref = O.df_jk_plain(Bp, nao, Cocc, D)
    assert np.array_equal(X[:, :, :nocc], X_emu)
    assert not X[:, :, nocc:].any()
    assert_k_matches_emulation(K, K_emu)
    assert O.rel_frobenius(J, J_ref) <= 1e-12
    assert O.rel_frobenius(K, K_ref) <= (1e-6 if s == 4 else 1e-10)
    assert np.array_equal(K, K.T)
    assert dfe.df_last_status() == 0


@pytest.mark.parametrize("s", [4, 7])
def test_emul_gemm_4096_sampled_rows_bitwise(dfe, gpu_ws, s):
    """Config-1 size 4096^3 in the launch configuration of the big GEMMs (cta_group::2 pair tiles,
    persistent grid, 128- or 64-byte K blocks).  The oracle emulates sampled rows of A against all of
    B: those rows of C must match bit for bit; the whole C within the tolerance of s slices."""
    n = 4096
    A, B = G.make_gemm_inputs(n, n, n, seed=21)
    C = torch.empty((n, n), dtype=torch.float64, device=DEV)
    dfe.df_emul_gemm_slices(dev(A), dev(B), C, n, n, n, s)
    torch.cuda.synchronize()
    Cg = C.cpu().numpy()
    rows = np.array([0, 1, 127, 128, 255, 256, 2047, 2048, 3000, 4095])
    eB, DB = O.split_operand(np.ascontiguousarray(B.T), s)
    eA, DA = O.split_operand(A[rows], s)
    assert np.array_equal(Cg[rows], O.emul_gemm_digits(eA, DA, eB, DB, s))
    err = O.rel_frobenius(Cg[rows], O.gemm_plain(A[rows], B))
    assert err <= (1e-6 if s == 4 else 1e-12), err
    assert dfe.df_last_status() == 0


@pytest.mark.parametrize("s", [4, 8])
def test_emul_gemm_16384_sampled_tiles_bitwise(dfe, gpu_ws, s):
    """the bit-exact integer check at the FULL size of BASELINE.json configs[1],
    16384^3, in the launch configuration bench.py --config gemm times.  At s = 8 the contraction exceeds
    KFLUSH(8) = 16352: the launch takes a second flush chunk of 32 elements on cta_group::2 pair tiles
    (the global read-modify-write of the running sum).  The operands are generated on the device
    (same distribution as make_gemm_inputs) and read back; the oracle emulates sampled rows of A against
    sampled columns of B over the full K -- first / last / boundary 128-tiles -- and those entries of C
    must match bit for bit."""
    n = 16384
    if s == 8:
        assert dfe.df_kflush(8) == 16352 < n
    if dfe.df_emul_gemm_workspace_bytes(n, n, n, s) > gpu_ws.view.numel():
        pytest.skip("workspace fixture too small")
    A, B = G.make_gemm_inputs_torch(n, n, n, seed=77, device=DEV)
    C = torch.empty((n, n), dtype=torch.float64, device=DEV)
    dfe.df_emul_gemm_slices(A, B, C, n, n, n, s)
    torch.cuda.synchronize()
    assert dfe.df_last_status() == 0
    rows = np.array([0, 1, 127, 128, 255, 256, 8191, 8192, 12345, 16383])
    cols = np.concatenate([np.arange(0, 130), np.arange(8190, 8194), np.arange(16384 - 130, 16384), [4099, 11111]])
    ti, tj = torch.from_numpy(rows).to(DEV), torch.from_numpy(cols).to(DEV)
    Ah = A.index_select(0, ti).cpu().numpy()                      # sampled rows of A, all of K
    Bh = B.index_select(1, tj).cpu().numpy()                      # all of K, sampled columns of B
    got = C.index_select(0, ti).index_select(1, tj).cpu().numpy()
    eA, DA = O.split_operand(Ah, s)
    eB, DB = O.split_operand(np.ascontiguousarray(Bh.T), s)       # one scale per column of B
    assert np.array_equal(got, O.emul_gemm_digits(eA, DA, eB, DB, s))
    err = O.rel_frobenius(got, O.gemm_plain(Ah, Bh))
    assert err <= (1e-6 if s == 4 else 1e-12), err
    del A, B, C


@pytest.mark.parametrize("flags", [8, 1 << 20, (1 << 20) | 8, 32 << 8, 64 << 8, 128 << 8, 1 << 23, (1 << 23) | 8, 1 << 24])
def test_emul_gemm_alternative_paths_bitwise(dfe, gpu_ws, flags):
    """The code paths the library does not pick by itself at these sizes (global read-modify-write
    of multi-pass tiles, one CTA per tile instead of cta_group::2 pairs, every K-block width, the
    staged 16-byte epilogue instead of 256-bit accesses) must give the same bits as the oracle's
    emulation."""
    m, n, k = 300, 260, 1500
    A, B = G.make_gemm_inputs(m, n, k, seed=31)
    Ad, Bd = dev(A), dev(B)
    dfe.lib.df_debug_set_gemm_flags(flags)
    try:
        for s in (1, 2, 3, 6, 8):  # s <= 2 takes 256-column tiles, s = 3 160-column tiles (bit 24: never)
            C = torch.empty((m, n), dtype=torch.float64, device=DEV)
            dfe.df_emul_gemm_slices(Ad, Bd, C, m, n, k, s)
            torch.cuda.synchronize()
            assert np.array_equal(C.cpu().numpy(), O.emul_gemm(A, B, s)), f"s={s}"
    finally:
        dfe.lib.df_debug_set_gemm_flags(0)


@pytest.mark.parametrize("flags", [4, 64, 4 | 8, 1 << 22, (1 << 22) | 64, 1 << 23, (1 << 23) | 4 | 8])
def test_jk_alternative_gemm5_paths(dfe, gpu_ws, flags):
    """GEMM(5) with one N tile (multi-pass), with the N halves on multicast CTA pairs instead of MMA
    pairs (bit 22), and with the halves on single CTAs (bit 6)."""
    nao, naux, nocc = 168, 38, 150
    Bp = G.make_B_packed(nao, naux, seed=13)
    Cocc = G.make_C_occ(nao, nocc, seed=13)
    D = G.make_density(Cocc)
    dfe.lib.df_debug_set_gemm_flags(flags)
    try:
        for s in (4, 5, 6):
            J, K, X, e6, ng = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
            K_emu, X_emu = O.emul_df_k(Bp, nao, Cocc, s, return_x=True)
            assert np.array_equal(X[:, :, :nocc], X_emu), f"s={s}"
            assert_k_matches_emulation(K, K_emu)
    finally:
        dfe.lib.df_debug_set_gemm_flags(0)


def test_two_contexts_two_streams_concurrent(dfe, gpu_ws):
    """one workspace per concurrent stream.  Two contexts, each with its own
    workspace, run different builds (and a GEMM) on two streams at the same time, several rounds
    interleaved; every result equals the serial one of the default context bit for bit.  The policy
    mode and the debug knobs belong to the context."""
    nao, nocc = 150, 20
    cases = []
    for seed, naux, s in ((61, 1100, 4), (62, 700, 6)):
        Bp = G.make_B_packed(nao, naux, seed=seed)
        Cocc = G.make_C_occ(nao, nocc, seed=seed)
        D = G.make_density(Cocc)
        Bd, Cd, Dd = dev(Bp), dev(Cocc), dev(D)
        J = torch.empty((nao, nao), dtype=torch.float64, device=DEV)
        K = torch.empty_like(J)
        dfe.df_jk_build_slices(Bd, nao, naux, Cd, nocc, Dd, s, J, K)
        cases.append((Bd, naux, Cd, Dd, s, J, K))
    A, B = G.make_gemm_inputs(300, 260, 1500, seed=63)
    Ad, Bgd = dev(A), dev(B)
    Cser = torch.empty((300, 260), dtype=torch.float64, device=DEV)
    dfe.df_emul_gemm(Ad, Bgd, Cser, 300, 260, 1500, 1e-8)
    torch.cuda.synchronize()
    nbytes = max(dfe.df_jk_workspace_bytes_blocks(nao, 1100, nocc, 6, 3), dfe.df_emul_gemm_workspace_bytes(300, 260, 1500, 8))
    ctxs = [dfe.Context(nbytes), dfe.Context(nbytes)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    try:
        outs = []
        for rnd in range(4):
            for i in (0, 1):
                Bd, naux, Cd, Dd, s, _, _ = cases[(i + rnd) % 2]
                J2 = torch.full((nao, nao), np.nan, dtype=torch.float64, device=DEV)
                K2 = torch.full_like(J2, np.nan)
                C2 = torch.full_like(Cser, np.nan)
                with torch.cuda.stream(streams[i]):
                    ctxs[i].jk_build_slices(Bd, nao, naux, Cd, nocc, Dd, s, J2, K2)
                    ctxs[i].emul_gemm(Ad, Bgd, C2, 300, 260, 1500, 1e-8)
                outs.append(((i + rnd) % 2, J2, K2, C2))
        torch.cuda.synchronize()
        for which, J2, K2, C2 in outs:
            assert torch.equal(J2, cases[which][5]) and torch.equal(K2, cases[which][6])
            assert torch.equal(C2, Cser)
        assert ctxs[0].last_status() == 0 and ctxs[1].last_status() == 0
        # per-context policy: nominal mode takes one slice less at this tolerance, guarded is unchanged
        ctxs[0].set_policy_mode(dfe.DF_MODE_NOMINAL)
        Cn, Cg = torch.empty_like(Cser), torch.empty_like(Cser)
        ctxs[0].emul_gemm(Ad, Bgd, Cn, 300, 260, 1500, 1e-8)
        ctxs[1].emul_gemm(Ad, Bgd, Cg, 300, 260, 1500, 1e-8)
        torch.cuda.synchronize()
        assert dfe.df_slices_for_tol(1e-8, dfe.DF_MODE_NOMINAL) < dfe.df_slices_for_tol(1e-8)
        assert np.array_equal(Cn.cpu().numpy(), O.emul_gemm(A, B, dfe.df_slices_for_tol(1e-8, dfe.DF_MODE_NOMINAL)))
        assert torch.equal(Cg, Cser)
        # per-context debug knobs: an alternative code path on one context only, same bits
        ctxs[1].set_debug_flags((1 << 20) | 8)
        ctxs[1].emul_gemm(Ad, Bgd, Cg, 300, 260, 1500, 1e-8)
        torch.cuda.synchronize()
        assert torch.equal(Cg, Cser)
    finally:
        for c in ctxs:
            c.close()


@pytest.mark.parametrize("s,nocc", [(3, 250), (4, 250), (3, 256), (4, 256)])
def test_gemm6_int32_guard_worst_case_digits_exact(dfe, gpu_ws, s, nocc):
    """The INT32 guard of GEMM(6)'s q-groups (R4/R5: s |g| nocc 2^14 < 2^31), pinned WITHOUT the
    oracle's grouping rule: every X^q_ia is the same value v whose balanced digits are the most
    negative a scaled operand can have, (-126, -128, ..., -128) (|x| 2^-e < 127/128 excludes a top
    digit beyond +-126 when the rest is -128), so every INT32 weight sum of every group is within 1 %
    of the largest a group of that length can reach: a group 2 % too long wraps around.  Whatever the
    grouping, K_ij = naux nocc sum_{t+u<=s+1} d_t d_u 2^(2e+2-8(t+u)), computed here in Python integers
    and exactly representable in FP64 at every partial sum -- K must equal it bit for bit."""
    nao, naux = 72, 600
    d = [-126] + [-128] * (s - 1)
    v = sum(dt * 256 ** (s - 1 - t) for t, dt in enumerate(d))  # an integer of 8 s bits: x = v, scale index 8 s - 1
    e = 8 * s - 1
    assert 0.5 <= abs(v) / 2.0 ** e < 127.0 / 128.0
    # B^q_i0 = v for every i and q, every other element 0; C_0a = 1, every other element 0  =>  X^q_ia = v
    Bp = np.zeros((nao * (nao + 1) // 2, naux))
    Bp[[i * (i + 1) // 2 for i in range(nao)], :] = float(v)
    Cocc = np.zeros((nao, nocc)); Cocc[0, :] = 1.0
    D = np.eye(nao)
    J, K, X, e6, ng = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
    assert ng >= 2 and np.array_equal(X[:, :, :nocc], np.full((naux, nao, nocc), float(v)))
    assert np.array_equal(e6, np.full((ng, nao), e))
    # per element: sum over the retained pairs, as an exact integer multiple of 2^(2e + 2 - 8(s + 1))
    unit = 2 * e + 2 - 8 * (s + 1)
    terms = [d[t] * d[u] * 2 ** (8 * (s + 1 - (t + 1) - (u + 1))) for t in range(s) for u in range(s) if t + u + 2 <= s + 1]
    total = sum(terms) * naux * nocc
    # every term is a multiple of 2^tz and the total below 2^(53 + tz): every partial sum, in any order, is exact
    tz = min((x & -x).bit_length() - 1 for x in terms)
    assert (total >> tz) < 2 ** 53 and unit >= 0
    # the worst weight sum of a maximal group really is at the edge of INT32: above 98 % of 2^31
    worst_pairs = max(sum(d[t] * d[w - 2 - t] for t in range(s) if 0 <= w - 2 - t < s) for w in range(2, s + 2))
    assert 0.98 * 2 ** 31 <= worst_pairs * (dfe.df_kflush(s) // nocc) * nocc < 2 ** 31
    assert np.array_equal(K, np.full((nao, nao), float(total * 2 ** unit)))
    assert np.array_equal(K, O.emul_df_k(Bp, nao, Cocc, s))
    assert dfe.df_last_status() == 0


@pytest.mark.parametrize("rule", ["energy_proxy", "density_change"])
def test_scf_sequence_every_step_within_its_tol(dfe, gpu_ws, rule):
    """The 12-step sequence of BASELINE.json configs[2] at a reduced size, under the schedule bench.py
    times (R11: dE_rel,k := eps_k^2) and under the density-change rule fed with the MEASURED
    ||D_k - D_{k-1}|| / ||D_k||: at EVERY step, not only the last, K is within the
    tolerance the schedule chose for that step of the oracle's plain FP64 K, and J within 1e-12."""
    from paper_2601_08077_b200 import policy

    nao, naux, nocc, seed = 160, 600, 24, 17
    Bp = G.make_B_packed(nao, naux, seed=seed)
    D0 = G.make_density(G.make_C_occ(nao, nocc, seed=seed))
    seq = G.make_scf_sequence(D0, nocc, 12, seed)
    if rule == "energy_proxy":
        sched = policy.schedule([eps * eps for eps, _, _ in seq])[:12]
    else:
        sched = policy.schedule_from_density_change(policy.measured_density_changes([Dk for _, Dk, _ in seq]))[:12]
    Bd = dev(Bp)
    J = torch.empty((nao, nao), dtype=torch.float64, device=DEV)
    K = torch.empty_like(J)
    used = []
    for (eps, Dk, Ck), (level, tol) in zip(seq, sched):
        dfe.df_jk_build(Bd, nao, naux, dev(Ck), nocc, dev(Dk), tol, J, K)
        torch.cuda.synchronize()
        J_ref, K_ref = O.df_jk_plain(Bp, nao, Ck, Dk)
        assert O.rel_frobenius(J.cpu().numpy(), J_ref) <= 1e-12, (rule, eps)
        err = O.rel_frobenius(K.cpu().numpy(), K_ref)
        assert err <= tol, (rule, eps, level, tol, err)
        used.append(dfe.df_slices_for_tol(tol))
    assert used == sorted(used) and used[0] < used[-1]  # precision only ever tightens, and it does
    assert dfe.df_last_status() == 0


def test_two_contexts_two_host_threads(dfe, gpu_ws):
    """Two contexts driven from two HOST threads (ctypes releases the GIL inside a call), same slice
    count, different contraction lengths: the row split's occupancy cap differs per call (the dynamic
    shared memory it asks for depends on `cols`), while the kernel attribute it is checked against is
    one per instantiation in the whole process.  Every call must succeed and give the serial bits,
    also with the per-class profiler recording from both threads."""
    import threading

    s = 4
    shapes = [(96, 64, 16384), (96, 64, 4096)]  # 148 SMs x cols x 8 bytes: 2 and 8 resident rows per SM
    ops = []
    for i, (m, n, k) in enumerate(shapes):
        A, B = G.make_gemm_inputs(m, n, k, seed=70 + i)
        Ad, Bd = dev(A), dev(B)
        Cser = torch.empty((m, n), dtype=torch.float64, device=DEV)
        dfe.df_emul_gemm_slices(Ad, Bd, Cser, m, n, k, s)
        ops.append((Ad, Bd, Cser))
    torch.cuda.synchronize()
    ctxs = [dfe.Context(dfe.df_emul_gemm_workspace_bytes(m, n, k, s)) for m, n, k in shapes]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    errors = []

    def work(i):
        m, n, k = shapes[i]
        Ad, Bd, Cser = ops[i]
        try:
            with torch.cuda.stream(streams[i]):
                for _ in range(200):
                    C2 = torch.full_like(Cser, np.nan)
                    ctxs[i].emul_gemm_slices(Ad, Bd, C2, m, n, k, s)
                streams[i].synchronize()
                if not torch.equal(C2, Cser):
                    errors.append((i, "bits differ"))
        except Exception as exc:  # DFError of a failed launch
            errors.append((i, repr(exc)))

    dfe.df_profile_enable(True)
    try:
        threads = [threading.Thread(target=work, args=(i,)) for i in (0, 1)]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        torch.cuda.synchronize()
        prof = dfe.df_profile_read()
    finally:
        dfe.df_profile_enable(False)
        for c in ctxs:
            c.close()
    assert not errors, errors
    assert prof["emul_gemm_i8"][1] == 400 and prof["split"][1] == 400, prof


@pytest.mark.parametrize("s", [3, 4, 6])
def test_jk_screened_input_bit_exact(dfe, gpu_ws, s):
    """on a B that decays away from the diagonal the
    build skips the K blocks of GEMM(5)'s left operand whose digits all vanish at s slices.  Only exact
    zeros are skipped, so X, the GEMM(6) scales and K are the DENSE oracle's, bit for bit; the counters
    show that blocks were skipped; with screening off (bit 25) and through a plan the bits are the same."""
    nao, naux, nocc = 600, 70, 40
    Bp = G.make_B_packed_screened(nao, naux, seed=70 + s, decay=0.6)
    Cocc = G.make_C_occ(nao, nocc, seed=70 + s)
    D = G.make_density(Cocc)
    dfe.df_screen_stats()
    J, K, X, e6, ng = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
    active, total = dfe.df_screen_stats()
    nblk = (naux * nao + 255) // 256
    assert total == nblk * 5 and 0 < active < 0.9 * total, (active, total)  # 5 K blocks of 128 columns
    K_emu, X_emu = O.emul_df_k(Bp, nao, Cocc, s, return_x=True)
    J_ref, K_ref = O.df_jk_plain(Bp, nao, Cocc, D)
    assert np.array_equal(X[:, :, :nocc], X_emu)
    groups = O.q_groups(naux, nocc, s)
    for g, (g0, g1) in enumerate(groups):
        Xrow = np.transpose(X_emu[g0:g1], (1, 0, 2)).reshape(nao, -1)
        assert np.array_equal(e6[g], O.scale_index(np.max(np.abs(Xrow), axis=1)))
    assert_k_matches_emulation(K, K_emu)
    assert O.rel_frobenius(J, J_ref) <= 1e-12
    assert dfe.df_last_status() == 0
    # screening off: every block is written, loaded and multiplied -- the same bits
    dfe.lib.df_debug_set_gemm_flags(1 << 25)
    try:
        J0, K0, X0, _, _ = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
        assert dfe.df_screen_stats() == (0, 0)
    finally:
        dfe.lib.df_debug_set_gemm_flags(0)
    assert np.array_equal(K0, K) and np.array_equal(X0, X) and np.array_equal(J0, J)
    # a plan made at 6 slices holds every block a build with s <= 6 reads
    Bd = dev(Bp)
    plan = dfe.Plan(Bd, nao, naux, 6)
    a6, t6 = dfe.df_screen_stats()
    assert t6 == total and active <= a6 < total  # the mask at 6 slices covers the mask at s
    J2 = torch.full((nao, nao), np.nan, dtype=torch.float64, device=DEV)
    K2 = torch.full_like(J2, np.nan)
    dfe.df_jk_build_planned_slices(plan, Bd, nao, naux, dev(Cocc), nocc, dev(D), s, J2, K2)
    torch.cuda.synchronize()
    assert np.array_equal(K2.cpu().numpy(), K) and np.array_equal(J2.cpu().numpy(), J)
    assert dfe.df_screen_stats()[0] == active
    plan.close()


def test_jk_dense_input_keeps_every_block(dfe, gpu_ws):
    """The configs' unstructured B: nothing is screened away."""
    cfg = G.CONFIGS["tiny"]
    Bp, Cocc, D = G.make_df_inputs(cfg)
    dfe.df_screen_stats()
    run_jk(dfe, Bp, cfg.nao, cfg.naux, Cocc, cfg.nocc, D, 4)
    active, total = dfe.df_screen_stats()
    assert active == total == (cfg.naux * cfg.nao + 255) // 256


def test_jk_screened_wide_mask_and_superblocks(dfe, gpu_ws):
    """Screening where the mask of a 256-row block spans two 32-bit words (nao = 4200: 33 K blocks of
    128 columns) and, separately, over several super-blocks (a minimum-size workspace: one 512-q block
    per launch, masks indexed from each super-block's first q).  X bit for bit against the dense oracle."""
    nao, naux, nocc, s = 4200, 6, 8, 3
    Bp = G.make_B_packed_screened(nao, naux, seed=81, decay=0.05)
    Cocc = G.make_C_occ(nao, nocc, seed=81)
    D = G.make_density(Cocc)
    dfe.df_screen_stats()
    J, K, X, e6, ng = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
    active, total = dfe.df_screen_stats()
    assert total == ((naux * nao + 255) // 256) * 33 and 0 < active < 0.6 * total, (active, total)
    K_emu, X_emu = O.emul_df_k(Bp, nao, Cocc, s, return_x=True)
    assert np.array_equal(X[:, :, :nocc], X_emu)
    assert_k_matches_emulation(K, K_emu)
    del Bp, X, X_emu

    nao, naux, nocc, s = 300, 1100, 12, 4
    Bp = G.make_B_packed_screened(nao, naux, seed=82, decay=0.5)
    Cocc = G.make_C_occ(nao, nocc, seed=82)
    D = G.make_density(Cocc)
    small = dfe.Workspace(dfe.df_jk_workspace_bytes(nao, naux, nocc, s))
    try:
        dfe.df_screen_stats()
        J, K, X, e6, ng = run_jk(dfe, Bp, nao, naux, Cocc, nocc, D, s)
        active, total = dfe.df_screen_stats()
    finally:
        small.close()
        dfe.df_set_workspace(gpu_ws.view)
    assert 0 < active < total
    K_emu, X_emu = O.emul_df_k(Bp, nao, Cocc, s, return_x=True)
    assert np.array_equal(X[:, :, :nocc], X_emu)
    assert_k_matches_emulation(K, K_emu)
    J_ref, _ = O.df_jk_plain(Bp, nao, Cocc, D)
    assert O.rel_frobenius(J, J_ref) <= 1e-12


def test_plan_of_screened_input_holds_every_scale_index(dfe, gpu_ws):
    """A plan made from a screened B into a buffer full of garbage: the scale index of EVERY row (q, i) is
    there (also of rows whose first K block is inactive and never written), and a planned build from it
    gives the bits of the plain build."""
    nao, naux, nocc, s = 768, 40, 24, 4  # a multiple of 256: a block of rows covers the same i for every q
    Bp = G.make_B_packed_screened(nao, naux, seed=91, decay=0.6)
    Cocc = G.make_C_occ(nao, nocc, seed=91)
    D = G.make_density(Cocc)
    Bd = dev(Bp)
    plan = dfe.Plan.__new__(dfe.Plan)
    plan.nao, plan.naux, plan.smax = nao, naux, 6
    nbytes = dfe.df_jk_plan_bytes(nao, naux, 6)
    plan.buf = torch.full((nbytes + 256,), 0x5A, dtype=torch.uint8, device=DEV)
    off = (-plan.buf.data_ptr()) % 256
    plan.view = plan.buf[off: off + nbytes]
    rc = dfe.lib.df_jk_plan_create(Bd.data_ptr(), nao, naux, 6, plan.view.data_ptr(), nbytes, None)
    assert rc == 0
    torch.cuda.synchronize()
    active, total = dfe.df_screen_stats()
    assert 0 < active < total
    rows = naux * nao
    r256 = lambda n: (n + 255) // 256 * 256
    e5_off = r256(rows * 4) + r256(((nao + 31) // 32) * ((nao + 31) // 32 + 1) // 2 * naux * 4)
    e5 = plan.view[e5_off: e5_off + rows * 4].view(torch.int32).cpu().numpy().reshape(naux, nao)
    for q in range(naux):
        Bq = O.unpack_sym(Bp[:, q], nao)
        assert np.array_equal(e5[q], O.scale_index(np.max(np.abs(Bq), axis=1))), q
    J = torch.empty((nao, nao), dtype=torch.float64, device=DEV)
    K = torch.empty_like(J)
    dfe.df_jk_build_slices(Bd, nao, naux, dev(Cocc), nocc, dev(D), s, J, K)
    J2, K2 = torch.full_like(J, np.nan), torch.full_like(K, np.nan)
    dfe.df_jk_build_planned_slices(plan, Bd, nao, naux, dev(Cocc), nocc, dev(D), s, J2, K2)
    torch.cuda.synchronize()
    assert torch.equal(J, J2) and torch.equal(K, K2)
    assert O.rel_frobenius(K.cpu().numpy(), O.emul_df_k(Bp, nao, Cocc, s)) <= 1e-14
