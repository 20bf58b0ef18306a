"""CPU-side checks of the C-ABI library: it loads without a GPU driver, exports every symbol
include/df_emul.h declares, and its host logic (policy, flush length, workspace sizing, argument
checks) matches the paper's Table 1 and the oracle's independent statement of the same rules."""
import ctypes
import math
import os
import re

import pytest

from oracle import df_oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "df_emul.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(df_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_all_exported(dfe):
    names = declared_symbols()
    assert "df_emul_gemm" in names and "df_jk_build" in names and len(names) >= 20
    raw = ctypes.CDLL(dfe.lib_path)
    for n in names:
        assert hasattr(raw, n), f"{n} declared in include/df_emul.h but not exported"
    # and the binding wraps every declared symbol under the same name
    assert set(names) == set(dfe.EXPORTS)


def test_library_has_no_driver_or_blas_dependency(dfe):
    import subprocess

    out = subprocess.run(["ldd", dfe.lib_path], capture_output=True, text=True).stdout
    for bad in ("libcuda.so", "libcublas", "libcudnn", "libtorch"):
        assert bad not in out


def test_policy_matches_table1(dfe):
    # tests/golden/table1_paper.txt is typed from PAPER.md:141-149
    rows = []
    for line in open(os.path.join(ROOT, "tests", "golden", "table1_paper.txt")):
        line = line.split("#")[0].strip()
        if line:
            rows.append(line.split())
    checked = 0
    for r in rows:
        try:
            m_emu, acc, splits = int(r[-3]), float(r[-2]), int(r[-1])
        except (ValueError, IndexError):
            continue
        assert dfe.df_slices_for_tol(acc, dfe.DF_MODE_NOMINAL) == splits == O.slices_from_mantissa_bits(m_emu)
        assert dfe.df_num_int8_gemms(splits) == splits * (splits + 1) // 2
        checked += 1
    assert checked >= 4


@pytest.mark.parametrize("mode", [0, 1])
def test_policy_agrees_with_oracle_statement(dfe, mode):
    name = "nominal" if mode == 0 else "guarded"
    for k in range(0, 70):
        for f in (1.0, 1.7, 3.3):
            tol = f * 2.0 ** (-k)
            assert dfe.df_slices_for_tol(tol, mode) == O.slices_for_tol(tol, name), (tol, mode)
    for tol in (1e-2, 1e-4, 1e-6, 1e-8, 1e-10, 1e-12, 1e-14, 1e-300, 0.5, 10.0):
        assert dfe.df_slices_for_tol(tol, mode) == O.slices_for_tol(tol, name)


def test_policy_rejects_bad_tol(dfe):
    for bad in (0.0, -1.0, float("nan")):
        with pytest.raises(dfe.DFError) as ei:
            dfe.df_slices_for_tol(bad)
        assert ei.value.code == -3
    with pytest.raises(dfe.DFError):
        dfe.df_slices_for_tol(1e-6, 7)


def test_kflush_guard(dfe):
    for s in range(1, 9):
        kf = dfe.df_kflush(s)
        assert kf == O.kflush(s) and kf % 32 == 0
        # INT32 guard: |P^(w)| <= (w-1) k 2^14 <= s k 2^14 < 2^31
        assert s * kf * (1 << 14) < (1 << 31) <= s * (kf + 32) * (1 << 14) + (1 << 20)
    with pytest.raises(dfe.DFError):
        dfe.df_kflush(9)


def test_workspace_sizes(dfe):
    prev = 0
    for s in range(1, 9):
        b = dfe.df_jk_workspace_bytes(1200, 4000, 150, s)
        assert b > prev
        prev = b
    # planes5 of one 512-q block dominate: s * 512 * nao * pitch(nao)
    b4 = dfe.df_jk_workspace_bytes(1200, 4000, 150, 4)
    assert b4 >= 4 * 512 * 1200 * 1216 and b4 < 8 << 30
    g = dfe.df_emul_gemm_workspace_bytes(1024, 1024, 1024, 3)
    assert g >= 2 * 3 * 1024 * 1024 and g < 2 * 3 * 1024 * 1024 + (1 << 20)
    assert dfe.df_plane_pitch(1200) == 1216 and dfe.df_plane_pitch(1) == 32
    with pytest.raises(dfe.DFError):
        dfe.df_jk_workspace_bytes(1200, 4000, 300, 4)  # nocc > 256 unsupported


def test_plan_sizes(dfe):
    """Plan = row maxima + scale indices (4 bytes each per (q, i)) + the maxima of the 32 x 32 tile
    pairs (4 bytes per pair and q; the screening mask's input) + smax planes of (q, i) rows padded
    to whole 128-byte lines; a planned build's workspace holds no GEMM(5) operand planes."""
    rows = 4000 * 1200
    pairs32 = 38 * 39 // 2  # ceil(1200 / 32) tiles per side
    r256 = lambda n: (n + 255) // 256 * 256  # every section starts on a 256-byte boundary
    assert dfe.df_jk_plan_bytes(1200, 4000, 6) == 2 * rows * 4 + r256(pairs32 * 4000 * 4) + 6 * rows * 1280
    assert dfe.df_jk_plan_bytes(100, 7, 1) == 2 * 2816 + 512 + 700 * 128  # 10 tile pairs x 7 q x 4 B -> 512
    w = dfe.df_jk_workspace_bytes_blocks(1200, 4000, 150, 4, 8)
    wp = dfe.df_jk_planned_workspace_bytes(1200, 4000, 150, 4, 8)
    assert 0 < wp <= w - 4 * rows * 1280
    for bad in ((0, 10, 4), (10, 0, 4), (20000, 10, 4)):
        with pytest.raises(dfe.DFError) as ei:
            dfe.df_jk_plan_bytes(*bad)
        assert ei.value.code == -2
    for smax in (0, 9):
        with pytest.raises(dfe.DFError) as ei:
            dfe.df_jk_plan_bytes(100, 10, smax)
        assert ei.value.code == -3


def test_plan_argument_errors_without_touching_a_device(dfe):
    lib = dfe.lib
    assert lib.df_jk_plan_create(None, 4, 4, 4, 256, 1 << 20, None) == -1
    assert lib.df_jk_plan_create(256, 4, 4, 4, None, 1 << 20, None) == -1
    assert lib.df_jk_plan_create(256, 0, 4, 4, 256, 1 << 20, None) == -2
    assert lib.df_jk_plan_create(256, 4, 4, 9, 256, 1 << 20, None) == -3
    assert lib.df_jk_plan_create(256, 4, 4, 4, 264, 1 << 20, None) == -7
    assert lib.df_jk_build_planned(None, 4, 1, 4, 4, 1, 1, 1, 1e-6, 1, 1, None) == -1
    assert lib.df_jk_build_planned_slices(256, 4, 1, 4, 4, 1, 1, 1, 5, 1, 1, None) == -3   # s > smax
    assert lib.df_jk_build_planned_slices(256, 0, 1, 4, 4, 1, 1, 1, 1, 1, 1, None) == -3   # smax out of range
    assert lib.df_jk_build_planned_slices(264, 4, 1, 4, 4, 1, 1, 1, 3, 1, 1, None) == -7   # misaligned plan
    assert lib.df_jk_build_planned_slices(256, 4, 1, 4, 4, 1, 300, 1, 3, 1, 1, None) == -2


def test_argument_errors_without_touching_a_device(dfe):
    lib = dfe.lib
    assert lib.df_emul_gemm(None, None, None, 4, 4, 4, 1e-6, None) == -1
    assert lib.df_emul_gemm_slices(1, 1, 1, 0, 4, 4, 3, None) == -2
    assert lib.df_emul_gemm_slices(1, 1, 1, 4, 4, 4, 9, None) == -3
    assert lib.df_emul_gemm(1, 1, 1, 4, 4, 4, float("nan"), None) == -3
    assert lib.df_jk_build(None, 4, 4, None, 1, None, 1e-6, None, None, None) == -1
    assert lib.df_jk_build_slices(1, 4, 4, 1, 300, 1, 3, 1, 1, None) == -2
    assert lib.df_set_workspace(None, 0) == 0


def test_no_cpu_fallback(dfe):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    # valid-looking arguments, no device: the library must refuse, not compute
    assert dfe.lib.df_emul_gemm_slices(256, 256, 256, 4, 4, 4, 3, None) == -5
    assert dfe.lib.df_set_workspace(256, 1 << 20) == -5
    assert dfe.lib.df_jk_plan_create(256, 4, 4, 4, 256, 1 << 20, None) == -5
    assert dfe.lib.df_jk_build_planned_slices(256, 4, 256, 4, 4, 256, 1, 256, 3, 256, 256, None) == -5


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2601_08077_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "df_oracle" not in text, f


def test_caller_schedule_matches_table1_and_oracle():
    from paper_2601_08077_b200 import policy

    # DESIGN.md R11: dE_rel,k = eps_k^2, eps_k = 10^(-k/2), k = 0..11
    dE = [10.0 ** (-k) for k in range(12)]
    got = policy.schedule(dE)
    ref = O.adaptive_schedule(dE)
    assert [lv for lv, _ in got] == [lv for lv, _ in ref]
    for (lv, tol), (_, m) in zip(got, ref):
        assert tol == 2.0 ** (-(m if m is not None else 52))
    levels = [lv for lv, _ in got[:12]]
    assert levels == sorted(levels, reverse=True)  # never revert
    # nominal splits 3 x7, 4 x3, 5 x2 over the 12 steps (R11)
    s_nom = [O.slices_for_tol(tol, "nominal") for _, tol in got[:12]]
    assert s_nom == [3] * 7 + [4] * 3 + [5] * 2
    # a noisy sequence never lowers the precision again
    lv = [l for l, _ in policy.schedule([1e-3, 1e-9, 1e-3, 1e-12, 1e-5, 1e-15, 1.0])]
    assert lv == [4, 4, 2, 2, 1, 1, 0, 0]  # 1e-9 < 5e-9 -> level 2; 1e-12 -> level 1


def test_context_entry_points_fail_loudly_without_a_device(dfe):
    """No GPU here: creating a context reports DF_ERR_DEVICE, a NULL context DF_ERR_NULL -- nothing
    falls back to the CPU."""
    import ctypes as C

    try:
        import torch

        if torch.cuda.is_available():
            pytest.skip("a CUDA device is present")
    except ImportError:
        pass
    h = C.c_void_p()
    assert dfe.lib.df_context_create(C.c_void_p(256), 1 << 20, C.byref(h)) == -5
    assert dfe.lib.df_context_create(None, 1 << 20, C.byref(h)) == -1
    assert dfe.lib.df_context_jk_build(None, None, 1, 1, None, 1, None, 1e-6, None, None, None) == -1
    assert dfe.lib.df_context_destroy(None) == -1


def test_density_change_schedule_is_the_energy_schedule_of_its_square():
    """policy.schedule_from_density_change (future work in the paper): dE_rel ~ dD_rel^2,
    then Table 1, monotone, lagged by one iteration, start level 4."""
    from paper_2601_08077_b200 import policy

    eps = [10.0 ** (-k / 2.0) for k in range(12)]
    got = policy.schedule_from_density_change(eps)
    assert got == policy.schedule([e * e for e in eps])
    levels = [lv for lv, _ in got][:12]
    assert levels == [4] * 7 + [3] * 3 + [2] * 2  # nominal splits 3 x 7, 4 x 3, 5 x 2 (R11)
    assert all(a >= b for a, b in zip(levels[:-1], levels[1:]))
    assert policy.level_for_density_change(1e-2) == 4 and policy.level_for_density_change(1e-8) == 0
    # the same levels as the oracle's independent statement of Table 1
    assert [lv for lv, _ in O.adaptive_schedule([e * e for e in eps])][:12] == levels


def test_measured_density_changes_of_the_synthetic_sequence():
    """The step-to-step change of D_k = D* + eps_k S_k (unit-norm S_k, eps_k = 10^(-k/2)) is
    sqrt(eps_k^2 + eps_{k-1}^2 - 2 eps_k eps_{k-1} <S_k, S_{k-1}>) / ||D_k||: close to
    sqrt(eps_k^2 + eps_{k-1}^2) / ||D*|| for independent S_k, and NOT eps_k itself; the schedule it
    drives is monotone and never looser than level 4."""
    import numpy as np

    from df_inputs import generators as G
    from paper_2601_08077_b200 import policy

    nao, nocc = 60, 8
    C0 = G.make_C_occ(nao, nocc, 5)
    D0 = G.make_density(C0)
    seq = G.make_scf_sequence(D0, nocc, 12, 5)
    dD = policy.measured_density_changes([Dk for _, Dk, _ in seq])
    assert dD[0] == 1.0 and len(dD) == 12
    for k in range(1, 12):
        want = np.hypot(seq[k][0], seq[k - 1][0]) / np.linalg.norm(D0)
        assert 0.8 * want <= dD[k] <= 1.25 * want, (k, dD[k], want)
    levels = [lv for lv, _ in policy.schedule_from_density_change(dD)][:12]
    assert levels[0] == levels[1] == 4 and all(a >= b for a, b in zip(levels[:-1], levels[1:]))


def test_ncu_table_is_rederivable_and_detects_stale_sources(tmp_path, monkeypatch):
    """profiles/ncu_kernels.csv (the counters bench.py quotes as roofline.traffic and tensor-pipe %) is
    what `bench.py --ncu-raw` distils from the committed raw ncu export, row for row; and the table is
    dropped (traffic null, traffic_stale true) as soon as the kernel sources differ from the ones it
    was captured on."""
    import csv
    import sys

    sys.path.insert(0, ROOT)
    import bench

    raw = os.path.join(ROOT, "profiles", "r03_ncu_full_raw.csv")
    committed = list(csv.DictReader(open(os.path.join(ROOT, bench.NCU_TABLE))))
    assert {(r["kernel_class"], r["s"]) for r in committed} >= {(c, str(s)) for c in ("gemm5_i8", "gemm6_i8", "jk_unpack_split")
                                                               for s in (4, 5, 6)}
    monkeypatch.setattr(bench, "NCU_TABLE", str(tmp_path / "t.csv"))
    bench.distill_ncu_raw([raw])
    again = list(csv.DictReader(open(tmp_path / "t.csv")))
    strip = lambda rows: [{k: v for k, v in r.items() if k != "sources_sha16"} for r in rows]
    assert strip(again) == strip(committed)
    table, stale = bench.ncu_table()
    assert not stale and len(table) == len(committed)  # distilled just now from these sources
    monkeypatch.setattr(bench, "kernel_sources_sha16", lambda: "0" * 16)
    table, stale = bench.ncu_table()
    assert stale
    assert bench.traffic_for_mix({}, ("gemm5_i8", "gemm6_i8"), [4, 5]) is None
