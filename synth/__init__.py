"""Seeded synthetic inputs for the transient F-statistic hot path.

This module is the ONE piece shared by the fp64 oracle (`oracle/`) and the CUDA
path (`paper_1805_05652_b200/`).  It holds no arithmetic of the method itself
(no window sums, no F-statistic, no marginalisation): it only manufactures atoms
{a2, b2, ab, Fa, Fb}, timestamps and grids with the shapes of the five
BASELINE.json configs.  See DESIGN.md "Input recipe".
"""
from .atoms import (  # noqa: F401
    TSFT,
    SIDEREAL_DAY,
    AtomSet,
    Grid,
    antenna_terms,
    gap_mask,
    make_atoms,
    make_detector_atoms,
    inject_exponential,
    inject_rectangular,
    template_seed,
    pack_atoms,
)
from .configs import CONFIGS, Workload, make_workload, tiny_workload  # noqa: F401
