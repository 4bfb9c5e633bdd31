"""CPU-side checks of the boundary (-m "not gpu"): libtfstat.so builds for sm_100a, loads
without a GPU, exports every symbol include/*.h declares, and validates arguments before
touching CUDA.  No compute calls are made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1805_05652_b200 import build, load_library

    build.build()  # nvcc cross-compiles without a GPU
    return load_library()


def declared_symbols(header):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return set(re.findall(r"\b(tfstat_[a-z_0-9]+)\s*\(", src))


def test_exports_every_declared_symbol(lib):
    names = declared_symbols("tfstat.h")
    assert {"tfstat_map", "tfstat_marginalise", "tfstat_search", "tfstat_search_host",
            "tfstat_workspace_bytes", "tfstat_count_terms", "tfstat_strerror",
            "tfstat_version", "tfstat_plan_info", "tfstat_validate_timestamps",
            "tfstat_map_general", "tfstat_merge_detectors"} <= names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/tfstat.h but not exported"
    assert lib.tfstat_version() == 200
    # the ALU micro-benchmarks live in a bench-only library of their own, not in the product
    from paper_1805_05652_b200 import load_probe_library

    probe = load_probe_library()
    pnames = declared_symbols("tfstat_probe.h")
    assert pnames == {"tfstat_probe_alu", "tfstat_probe_direct_loop"}
    for n in pnames:
        assert hasattr(probe, n)
        assert not hasattr(lib, n), f"{n} must not ship inside libtfstat.so"


def test_opts_struct_size_and_plan_info(lib):
    """tfstat_opts starts with its own size, so the struct can grow: a shorter (older) struct is
    accepted and the missing fields take defaults; size 0 / reserved fields set are EINVAL.
    tfstat_plan_info reports the kernel, tile and workspace tfstat_search would use."""
    import paper_1805_05652_b200 as pkg
    import paper_1805_05652_b200.binding as b

    fake = C.c_void_p(0x1000)
    grid = [0, 1800, 4, 3600, 1800, 4]
    o = b._Opts()
    assert o.struct_size == C.sizeof(b._Opts) == 56
    o.struct_size = 0
    assert lib.tfstat_search(fake, 70, 10, fake, 10, 1, 1, *grid, fake, None, None, fake, 1 << 20,
                             None, C.byref(o)) == -1
    assert lib.tfstat_workspace_bytes(1, 10, 1, *grid, C.byref(o)) == 0
    o = b._Opts()
    o.reserved0 = 1
    assert lib.tfstat_workspace_bytes(1, 10, 1, *grid, C.byref(o)) == 0
    # an "old" caller that only knows the fields up to exp_method: exp_method is honoured, a
    # tile_c lying beyond its struct_size is ignored
    g = G(0, 1800, 96, 43200, 1800, 1417)
    o = b._Opts()
    o.exp_method, o.tile_c = pkg.EXP_DIRECT, 2
    p = b._Plan()
    p.struct_size = C.sizeof(b._Plan)
    assert lib.tfstat_plan_info(1, 2880, 4096, *b._grid_args(g), C.byref(o), C.byref(p)) == 0
    assert (p.kernel, p.tile_c) == (1, 2)
    o.struct_size = 12
    assert lib.tfstat_plan_info(1, 2880, 4096, *b._grid_args(g), C.byref(o), C.byref(p)) == 0
    assert (p.kernel, p.tile_c, p.tile_nt) == (1, 8, 128)  # config 4: the headline tile
    assert p.n_ctas == 4096 * 12 * 12 and p.n_launches == 4
    assert p.workspace_bytes == lib.tfstat_workspace_bytes(1, 2880, 4096, *b._grid_args(g), C.byref(o))
    # defaults: the sliding form; config 1: the one-launch rect kernel; invalid shapes: errors
    info = pkg.plan_info(pkg.EXP, 2880, 4096, g)
    # (tile_c of the sliding form: templates per CTA of the slide kernel + 10 x (10 RT + TPC) of the
    # per-tau window-sum kernel, which here only has the 109 smallest tau values left: two per
    # thread x 2 templates; 4 templates per CTA in the slide kernel; 6 launches: bounds, pack,
    # per-tau window sums, grouped window sums, slide, finalize)
    assert info["kernel_name"] == "exp_slide" and info["tile_c"] == 224 and info["n_launches"] == 6
    # 1000 + ...: every window sum by the per-tau kernel
    info = pkg.plan_info(pkg.EXP, 2880, 4096, g, tile=(1000, 0, 0))
    assert info["tile_c"] == 424 and info["n_launches"] == 5
    assert pkg.plan_info(pkg.RECT, 48, 1, G(0, 1800, 24, 1800, 1800, 24))["kernel_name"] == "rect_small"
    big = pkg.plan_info(pkg.RECT, 13140, 1, G(0, 1800, 17520, 43200, 43200, 720))
    assert big["kernel_name"] == "rect_run" and big["lattice_J"] == 17519 + 719 * 24 + 1
    with pytest.raises(pkg.TfstatError):
        pkg.plan_info(pkg.EXP, 10, 1, G(0, 1800, 0, 3600, 1800, 4))
    assert lib.tfstat_plan_info(1, 10, 1, *grid, None, None) == -1


def test_sass_is_sm100a():
    import shutil
    import subprocess

    from paper_1805_05652_b200 import lib_path

    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not on PATH")
    out = subprocess.run(["cuobjdump", "-lelf", lib_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out and "sm_90" not in out


def test_result_struct_layout():
    from paper_1805_05652_b200 import RESULT_DTYPE

    assert RESULT_DTYPE.itemsize == 20
    assert [RESULT_DTYPE.fields[k][1] for k in ("max2F", "m", "n", "logB", "n_valid")] == [
        0, 4, 8, 12, 16]


class G:
    def __init__(self, *a):
        (self.t0_min, self.dt0, self.N_t0, self.tau_min, self.dtau, self.N_tau) = a


def test_workspace_bytes_and_validation(lib):
    import paper_1805_05652_b200 as pkg

    g = G(0, 1800, 96, 43200, 1800, 1417)
    small = pkg.workspace_bytes(pkg.EXP, 2880, 1, g)
    big = pkg.workspace_bytes(pkg.EXP, 2880, 4096, g)
    assert 0 < small < big < 1 << 30
    assert pkg.workspace_bytes(pkg.RECT, 13140, 1, G(0, 1800, 17520, 43200, 43200, 720)) > 13141 * 64
    for bad in (G(0, 1800, 0, 3600, 1800, 4), G(0, 1800, 4, 0, 1800, 4), G(0, 0, 4, 3600, 1800, 4),
                G(0, 1800, 4, 3600, 0, 4), G(0, 1, 1 << 16, 1, 1, 1 << 16)):
        with pytest.raises(pkg.TfstatError):
            pkg.workspace_bytes(pkg.EXP, 10, 1, bad)
    with pytest.raises(pkg.TfstatError):
        pkg.workspace_bytes(7, 10, 1, g)


def test_error_codes_before_any_cuda_call(lib):
    """Validation happens on the host before anything is enqueued, so fake non-null pointers
    are never dereferenced here."""
    fake = C.c_void_p(0x1000)
    grid = [0, 1800, 4, 3600, 1800, 4]
    opts = None
    # null required pointer
    assert lib.tfstat_search(None, 70, 10, fake, 10, 1, 1, *grid, fake, None, None, fake, 1 << 20,
                             None, opts) == -1
    # neither results nor maps requested
    assert lib.tfstat_search(fake, 70, 10, fake, 10, 1, 1, *grid, None, None, None, fake, 1 << 20,
                             None, opts) == -1
    # ld < n_atoms
    assert lib.tfstat_search(fake, 70, 9, fake, 10, 1, 1, *grid, fake, None, None, fake, 1 << 20,
                             None, opts) == -1
    # unknown window
    assert lib.tfstat_search(fake, 70, 10, fake, 10, 1, 5, *grid, fake, None, None, fake, 1 << 20,
                             None, opts) == -1
    # workspace too small / missing
    assert lib.tfstat_search(fake, 70, 10, fake, 10, 1, 1, *grid, fake, None, None, fake, 8,
                             None, opts) == -2
    assert lib.tfstat_search(fake, 70, 10, fake, 10, 1, 1, *grid, fake, None, None, None, 1 << 20,
                             None, opts) == -2
    # t0_max + 3 tau_max beyond int32
    ov = [0, 1800, 4, 700_000_000, 1_000_000, 40]
    assert lib.tfstat_search(fake, 70, 10, fake, 10, 1, 1, *ov, fake, None, None, fake, 1 << 20,
                             None, opts) == -4
    assert lib.tfstat_map(fake, 10, fake, 10, 0, *grid, None, None, fake, 1 << 20, None, opts) == -1
    assert lib.tfstat_marginalise(None, None, 4, 4, fake, fake, 1 << 20, None, None) == -1
    assert lib.tfstat_marginalise(fake, None, 4, 4, fake, fake, 0, None, None) == -2
    # a workspace that is not 16-byte aligned is an error, not a device fault
    assert lib.tfstat_marginalise(fake, None, 4, 4, fake, C.c_void_p(0x1004), 1 << 20, None,
                                  None) == -2
    # the no-allocation variant: null pointers, empty maps, maps beyond its stated maximum
    assert lib.tfstat_marginalise_static(None, None, 4, 4, fake, None) == -1
    assert lib.tfstat_marginalise_static(fake, None, 4, 4, None, None) == -1
    assert lib.tfstat_marginalise_static(fake, None, 0, 4, fake, None) == -1
    assert lib.tfstat_marginalise_static(fake, None, 65536, 32768, fake, None) == -1
    assert lib.tfstat_marginalise_static_max_cells() == 2**31 - 1
    # tfstat_validate_timestamps / tfstat_count_terms: null pointers, empty input
    assert lib.tfstat_validate_timestamps(None, 10, fake, None, None) == -1
    assert lib.tfstat_validate_timestamps(fake, 10, None, None, None) == -1
    assert lib.tfstat_validate_timestamps(fake, 0, fake, None, None) == -1
    assert lib.tfstat_count_terms(None, 10, 1, *grid, fake, fake, 1 << 20, None, None) == -1
    assert lib.tfstat_strerror(-2).decode().startswith("workspace")
    # rect_method / exp_method out of range
    import paper_1805_05652_b200.binding as b
    o = b._Opts()
    o.rect_method = 3
    assert lib.tfstat_search(fake, 70, 10, fake, 10, 1, 0, *grid, fake, None, None, fake, 1 << 20,
                             None, C.byref(o)) == -1
    o = b._Opts()
    o.exp_method = 9
    assert lib.tfstat_search(fake, 70, 10, fake, 10, 1, 1, *grid, fake, None, None, fake, 1 << 20,
                             None, C.byref(o)) == -1
    # tfstat_map_general: null window, bad kind, empty support, table missing, workspace
    w = b._Window()
    w.kind, w.support_num, w.support_den = 1, 3, 1
    args = lambda win, ws=fake, nws=1 << 20: (fake, 10, fake, 10, win, fake, 4, fake, 4, fake, None,  # noqa: E731
                                              None, ws, nws, None, None)
    assert lib.tfstat_map_general(*args(None)) == -1
    assert lib.tfstat_map_general(*args(C.byref(w), None)) == -2
    assert lib.tfstat_map_general(*args(C.byref(w), fake, 8)) == -2
    w.kind = 7
    assert lib.tfstat_map_general(*args(C.byref(w))) == -1
    w.kind, w.support_num = 1, 0
    assert lib.tfstat_map_general(*args(C.byref(w))) == -1
    w.kind, w.support_num, w.n_table = 2, 1, 0
    assert lib.tfstat_map_general(*args(C.byref(w))) == -1
    assert lib.tfstat_general_workspace_bytes(0, 4) == 0
    assert lib.tfstat_general_workspace_bytes(4, 300) == 256 * ((32 * 4 * 3 + 255) // 256)
    # tfstat_merge_detectors: n_det out of range, null arrays, ld < n
    pa = (C.c_void_p * 1)(0x1000)
    i64 = (C.c_int64 * 1)(70)
    ld = (C.c_int64 * 1)(10)
    n = (C.c_int32 * 1)(10)
    assert lib.tfstat_merge_detectors(pa, i64, ld, pa, n, 0, 1, fake, 10, fake, 70, 10, None, None) == -1
    assert lib.tfstat_merge_detectors(pa, i64, ld, pa, n, 9, 1, fake, 10, fake, 70, 10, None, None) == -1
    assert lib.tfstat_merge_detectors(None, i64, ld, pa, n, 1, 1, fake, 10, fake, 70, 10, None, None) == -1
    assert lib.tfstat_merge_detectors(pa, i64, ld, pa, n, 1, 1, fake, 10, fake, 70, 9, None, None) == -1
    ld[0] = 9
    assert lib.tfstat_merge_detectors(pa, i64, ld, pa, n, 1, 1, fake, 10, fake, 70, 10, None, None) == -1
    # tfstat_search_host: null host pointers, misaligned scratch
    assert lib.tfstat_search_host(None, 70, 10, fake, 10, 1, 1, *grid, fake, None, None, 0,
                                  None) == -1
    assert lib.tfstat_search_host(fake, 70, 10, fake, 10, 1, 1, *grid, fake, None,
                                  C.c_void_p(0x1001), 1 << 20, None) == -2
    assert lib.tfstat_search_host_scratch_bytes(70, 10, 0, 1, *grid, 0, None) == 0
    assert lib.tfstat_search_host_scratch_bytes(70, 10, 5, 1, *grid, 1, None) > 5 * 70 * 4 * 2


def test_missing_library_fails_loudly(monkeypatch):
    import paper_1805_05652_b200.binding as b

    monkeypatch.setattr(b, "_lib", None)
    monkeypatch.setattr(b, "_LIB_PATH", "/nonexistent/libtfstat.so")
    with pytest.raises(b.TfstatError, match="no CPU fallback"):
        b.load_library()


def test_product_never_imports_oracle():
    """The CUDA path and the oracle share no code and neither imports the other."""
    pkg_dir = os.path.join(ROOT, "paper_1805_05652_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "tfstat_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1805_05652_b200" not in src.replace("paper_1805_05652_b200/", ""), f
            assert not re.search(r"^\s*(import|from)\s+paper_1805_05652_b200\b", src, flags=re.M), f
