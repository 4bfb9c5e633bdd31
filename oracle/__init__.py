"""fp64 CPU oracle for the transient F-statistic map -- TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this package.  It shares nothing with the
CUDA path (`paper_1805_05652_b200/`), which must never import it.

The arithmetic lives in `tfstat_oracle.c` (plain C, fp64, the paper's
definitions cell by cell); this file only compiles it with gcc and marshals
numpy arrays through ctypes.
"""
from .binding import (  # noqa: F401
    EXP,
    RECT,
    OracleResult,
    build,
    cells,
    map2F,
    marginalise,
    num_threads,
    search,
)
