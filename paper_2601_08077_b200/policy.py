"""Caller side of the tolerance policy (row H0 of SURVEY.md 8(a)): the adaptive schedule of
PAPER.md:132-151.  After SCF iteration i the caller computes dE_rel,i (Eq. 11),
looks it up in Table 1 and passes the resulting emulation accuracy as `tol`
to df_jk_build for iteration i+1; precision never goes back down and iteration 0 starts at
m_emu = 23.  The library then maps tol -> slices (df_slices_for_tol).

Host-only, no arithmetic of the method itself; the table is typed from the paper.
"""
from __future__ import annotations

# (lower bound of dE_rel, emulation level, mantissa bits m_emu)
TABLE1 = ((2e-6, 4, 23), (5e-9, 3, 31), (2e-11, 2, 39), (7e-14, 1, 47))
# Level 0 is "standard FP64" in the paper (2.2e-16).  The library has no native-FP64 GEMM
# (DESIGN.md section 8): level 0 asks for tol = 2^-52, which the guarded policy runs with s = 8 slices.
# That is at least as accurate as an FP64 GEMM (tests/test_oracle_emulation.py pins it against a long-double
# reference: 4e-17 against 4e-16 rel-F) and on B200 also the faster of the two: an s = 7..8 emulation sustains
# more effective FP64 FLOP/s on the INT8 tensor pipe than the chip's native FP64 peak.
M_EMU_OF_LEVEL = {4: 23, 3: 31, 2: 39, 1: 47, 0: 52}
START_LEVEL = 4


def level_for(dE_rel: float) -> int:
    """Emulation level for the NEXT iteration given this iteration's relative energy change."""
    for lo, level, _ in TABLE1:
        if dE_rel >= lo:
            return level
    return 0


def tol_of_level(level: int) -> float:
    """Table 1's "Emu. Relative Accuracy" column: 2^-m_emu."""
    return 2.0 ** (-M_EMU_OF_LEVEL[level])


class AdaptiveTolerance:
    """tol for each SCF iteration; feed it dE_rel after every iteration."""

    def __init__(self):
        self.level = START_LEVEL

    @property
    def tol(self) -> float:
        return tol_of_level(self.level)

    def update(self, dE_rel: float) -> float:
        self.level = min(self.level, level_for(abs(dE_rel)))  # never revert
        return self.tol


def level_for_density_change(dD_rel: float) -> int:
    """Emulation level for the NEXT iteration from the relative change of the density matrix,
    ||D_k - D_{k-1}||_F / ||D_k||_F (the paper names a density-driven choice as future work).
    The energy is stationary in the density, so its error is second order in the density error
    (R11): dE_rel ~ dD_rel^2, looked up in Table 1 like a measured energy change."""
    return level_for(dD_rel * dD_rel)


def schedule_from_density_change(dD_rels):
    """[(level, tol)] like `schedule`, driven by the density changes instead of the energy changes."""
    return schedule([d * d for d in dD_rels])


def measured_density_changes(densities):
    """dD_rel,k = ||D_k - D_{k-1}||_F / ||D_k||_F of consecutive density matrices (NumPy arrays), the
    input of schedule_from_density_change.  Iteration 0 has no predecessor: its change is reported as
    1.0, which keeps the start level."""
    import numpy as np

    out = [1.0]
    for prev, cur in zip(densities[:-1], densities[1:]):
        out.append(float(np.linalg.norm(cur - prev) / np.linalg.norm(cur)))
    return out


def schedule(dE_rels):
    """[(level, tol)] for iterations 0..len(dE_rels): iteration i+1 uses dE_rel of iteration i."""
    a = AdaptiveTolerance()
    out = [(a.level, a.tol)]
    for d in dE_rels:
        a.update(d)
        out.append((a.level, a.tol))
    return out
