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


def declared_symbols():
    names = set()
    for h in ("tfstat.h", "tfstat_probe.h"):
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(tfstat_[a-z_0-9]+)\s*\(", src))
    return names


def test_exports_every_declared_symbol(lib):
    names = declared_symbols()
    assert {"tfstat_map", "tfstat_marginalise", "tfstat_search", "tfstat_search_host",
            "tfstat_workspace_bytes", "tfstat_count_terms", "tfstat_strerror",
            "tfstat_version", "tfstat_probe_alu"} <= names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/ but not exported"
    assert lib.tfstat_version() == 100


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
    assert lib.tfstat_marginalise(None, None, 4, 4, fake, fake, 1 << 20, None) == -1
    assert lib.tfstat_marginalise(fake, None, 4, 4, fake, fake, 0, None) == -2
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
    assert lib.tfstat_merge_detectors(pa, i64, ld, pa, n, 0, 1, fake, 10, fake, 70, 10, None) == -1
    assert lib.tfstat_merge_detectors(pa, i64, ld, pa, n, 9, 1, fake, 10, fake, 70, 10, None) == -1
    assert lib.tfstat_merge_detectors(None, i64, ld, pa, n, 1, 1, fake, 10, fake, 70, 10, None) == -1
    assert lib.tfstat_merge_detectors(pa, i64, ld, pa, n, 1, 1, fake, 10, fake, 70, 9, None) == -1
    ld[0] = 9
    assert lib.tfstat_merge_detectors(pa, i64, ld, pa, n, 1, 1, fake, 10, fake, 70, 10, None) == -1
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
