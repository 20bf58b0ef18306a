"""Seeded synthetic inputs for the DF J/K hot path (arXiv 2601.08077).

This module is the ONLY code shared by the CPU oracle's tests and the CUDA
path's tests/bench.  It holds none of the method's arithmetic: no slicing, no
scale indices, no contractions -- only random inputs with the shapes and
magnitude distributions BASELINE.json's configs describe (which stand in for
the paper's Table 3 molecules; the molecules, basis sets and
PySCF are not available here).
"""
from .generators import (  # noqa: F401
    CONFIGS,
    DFConfig,
    npair,
    pair_index,
    make_B_packed,
    make_C_occ,
    make_density,
    make_df_inputs,
    make_gemm_inputs,
    make_gemm_inputs_torch,
    make_scf_sequence,
    occ_from_density,
    make_B_packed_torch,
)
