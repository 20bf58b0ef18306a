"""Pins for the tol -> slices policy and the Table 1 schedule -- CPU only.
Expected values come from the paper's Table 1 (tests/golden/table1_paper.txt,
PAPER.md:141-147) and its formulas."""
import math
import os

import pytest

import oracle as O


def _table1(golden_dir):
    rows = []
    with open(os.path.join(golden_dir, "table1_paper.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            lo, level, m, acc, splits = line.split()
            rows.append((float(lo), int(level), None if m == "-" else int(m), float(acc), int(splits)))
    return rows


def test_table1_rows_closed_form(golden_dir):
    rows = _table1(golden_dir)
    assert [r[1] for r in rows] == [4, 3, 2, 1, 0]
    for lo, level, m, acc, splits in rows[:-1]:
        # s = ceil((m_emu + 1)/8)
        assert O.slices_from_mantissa_bits(m) == splits
        # printed accuracy = 2^-m_emu to 2 significant figures
        assert float(f"{2.0 ** -m:.1e}") == acc
        # nominal policy reproduces the paper's split count from its accuracy column
        assert O.slices_for_tol(acc, "nominal") == splits
    assert float(f"{2.0 ** -52:.1e}") == rows[-1][3]
    # "10 or more INT8 GEMMs" at 4 splits
    assert O.num_int8_gemms(4) == 10 and O.num_int8_gemms(3) == 6 and O.num_int8_gemms(6) == 21


def test_table1_bands(golden_dir):
    rows = _table1(golden_dir)
    for (lo, level, m, _, _), nxt in zip(rows[:-1], rows[1:]):
        assert O.table1_level(lo) == (level, m)
        assert O.table1_level(lo * 1.5) == (level, m)
        assert O.table1_level(lo * (1 - 1e-9))[0] == nxt[1]
    assert O.table1_level(1.0) == (4, 23)
    assert O.table1_level(1e-15) == (0, None)


def test_schedule_monotone_and_lagged():
    # dE_rel of iteration i selects iteration i+1; iteration 0 is m_emu = 23
    dE = [1e-2, 1e-7, 1e-4, 1e-10, 1e-9, 1e-12, 1e-15, 1e-3]
    sched = O.adaptive_schedule(dE)
    assert len(sched) == len(dE) + 1
    assert sched[0] == (4, 23)
    assert [lv for lv, _ in sched] == [4, 4, 3, 3, 2, 2, 1, 0, 0]
    levels = [lv for lv, _ in sched]
    assert all(a >= b for a, b in zip(levels[:-1], levels[1:]))  # never revert


def test_synthetic_scf_sequence_slices():
    # proxy dE_rel,k = eps_k^2, eps_k = 10^(-k/2), 12 steps
    dE = [(10.0 ** (-k / 2.0)) ** 2 for k in range(12)]
    sched = O.adaptive_schedule(dE)[:12]
    splits = [O.slices_from_mantissa_bits(m) for _, m in sched]
    assert splits == [3] * 7 + [4] * 3 + [5] * 2


def test_guarded_rule_values():
    want = {1e-2: 2, 1e-4: 3, 1e-6: 4, 1e-8: 5, 1e-10: 6, 1e-12: 6, 1e-14: 7, 1e-16: 8, 1e-30: 8, 0.9: 1}
    for tol, s in want.items():
        assert O.slices_for_tol(tol, "guarded") == s
        assert O.slices_for_tol(tol, "guarded") == min(8, max(1, math.ceil((math.log2(1 / tol) + 7) / 8)))
        assert O.slices_for_tol(tol, "guarded") >= O.slices_for_tol(tol, "nominal") or tol > 0.5
    with pytest.raises(ValueError):
        O.slices_for_tol(0.0)
    with pytest.raises(ValueError):
        O.slices_for_tol(float("nan"))
