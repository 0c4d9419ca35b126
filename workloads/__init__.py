"""Seeded synthetic input generators for the five BASELINE.json workloads (and small test variants).

This module serves BOTH the CPU oracle (oracle/) and the CUDA path (paper_1708_03621_b200/); it
imports neither and holds none of the method's arithmetic (no FFT, no operator, no basis rule): it
only produces input DATA -- lattice, k-points, cutoffs, box sizes, band coefficients C, the local
potential V_loc, projectors P and the coupling D.  The G-sphere `iG` that P depends on is passed IN
by the caller (from whichever side it is driving).  Recipe: DESIGN.md section 4 (= SURVEY.md 8(d)).
"""
from .configs import CONFIGS, TEST_CONFIGS, get_config  # noqa: F401
from .generate import (atoms_fractional, make_bands, make_D, make_inputs, make_projectors,  # noqa: F401
                       make_vloc, lattice)
