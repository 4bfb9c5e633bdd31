"""paper_1805_05652_b200 -- the transient F-statistic map (Keitel & Ashton 2018,
arXiv:1805.05652) as hand-written CUDA for NVIDIA B200 (sm_100a).

The product is `libtfstat.so` (C ABI in `include/tfstat.h`, sources in `csrc/`).  This Python
package is a thin ctypes binding with the same call names: argument marshalling only, every
step of the path runs in the CUDA kernels.  There is no CPU fallback: importing the binding
without the built library raises.
"""
from .binding import (  # noqa: F401
    EXP,
    EXP_AUTO,
    EXP_DIRECT,
    EXP_SCAN,
    RECT,
    RESULT_DTYPE,
    TABLE,
    TfstatError,
    count_terms,
    lib_path,
    load_library,
    load_probe_library,
    plan_info,
    probe_alu,
    probe_direct_loop,
    search_host_scratch_bytes,
    tfstat_map,
    tfstat_map_general,
    tfstat_marginalise,
    tfstat_marginalise_static,
    tfstat_merge_detectors,
    tfstat_search,
    tfstat_search_host,
    validate_timestamps,
    workspace_bytes,
)
from .shard import gather_results, template_shard  # noqa: F401,E402
