"""ctypes binding of libtfstat.so (include/tfstat.h).  Argument marshalling only.

PyTorch is used for device memory and streams; every step of the hot path runs inside the
CUDA kernels of csrc/.  There is no CPU fallback: a missing library raises TfstatError.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np
import torch

RECT, EXP, TABLE = 0, 1, 2
EXP_AUTO, EXP_DIRECT, EXP_SCAN = 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtfstat.so")
_PROBE_LIB_PATH = os.path.join(_HERE, "libtfstat_probe.so")
_lib = None
_probe_lib = None
N_STATS = 8  # TFSTAT_N_STATS
STAT_NAMES = ("terms_window", "terms_enter", "terms_leave", "terms_resum", "cells", "redo64",
              "terms_moment")
KERNEL_NAMES = {1: "exp_direct", 2: "exp_slide", 3: "rect_small", 4: "rect_run", 5: "rect_cells",
                6: "rect_tile"}

# tfstat_result, 20 bytes (include/tfstat.h)
RESULT_DTYPE = np.dtype([("max2F", "<f4"), ("m", "<i4"), ("n", "<i4"), ("logB", "<f4"),
                         ("n_valid", "<i4")])


class TfstatError(RuntimeError):
    pass


class _Opts(C.Structure):
    """tfstat_opts (include/tfstat.h); struct_size is filled in by __init__."""
    _fields_ = [("struct_size", C.c_uint32), ("min_atoms", C.c_int32), ("exp_method", C.c_int32),
                ("rect_method", C.c_int32), ("tile_c", C.c_int32), ("tile_nt", C.c_int32),
                ("seg_len", C.c_int32), ("reserved0", C.c_int32), ("ev_main_begin", C.c_void_p),
                ("ev_main_end", C.c_void_p), ("stats", C.c_void_p)]

    def __init__(self, *a, **k):
        super().__init__(*a, **k)
        self.struct_size = C.sizeof(_Opts)


class _Plan(C.Structure):
    """tfstat_plan (include/tfstat.h)."""
    _fields_ = [("struct_size", C.c_uint32), ("kernel", C.c_int32), ("tile_c", C.c_int32),
                ("tile_nt", C.c_int32), ("seg_len", C.c_int32), ("n_segs", C.c_int32),
                ("n_launches", C.c_int32), ("lattice_J", C.c_int32), ("n_ctas", C.c_int64),
                ("workspace_bytes", C.c_uint64)]


class _Window(C.Structure):
    _fields_ = [("kind", C.c_int32), ("support_num", C.c_int32), ("support_den", C.c_int32),
                ("n_table", C.c_int32), ("table", C.c_void_p)]


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen libtfstat.so; raises if it has not been built (python -m paper_1805_05652_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise TfstatError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_1805_05652_b200.build` "
            "(nvcc, sm_100a).  libtfstat has no CPU fallback.")
    lib = C.CDLL(_LIB_PATH)
    i32, i64, vp, sz = C.c_int32, C.c_int64, C.c_void_p, C.c_size_t
    grid = [i32] * 6
    op = C.POINTER(_Opts)
    lib.tfstat_version.restype = C.c_int
    lib.tfstat_strerror.restype = C.c_char_p
    lib.tfstat_strerror.argtypes = [C.c_int]
    lib.tfstat_last_cuda_error.restype = C.c_int
    lib.tfstat_workspace_bytes.restype = sz
    lib.tfstat_workspace_bytes.argtypes = [C.c_int, i32, i32] + grid + [op]
    lib.tfstat_map.argtypes = [vp, i64, vp, i32, C.c_int] + grid + [vp, vp, vp, sz, vp, op]
    lib.tfstat_marginalise_workspace_bytes.restype = sz
    lib.tfstat_marginalise_workspace_bytes.argtypes = [i32, i32]
    lib.tfstat_marginalise.argtypes = [vp, vp, i32, i32, vp, vp, sz, vp, op]
    lib.tfstat_marginalise_static_max_cells.restype = sz
    lib.tfstat_marginalise_static_max_cells.argtypes = []
    lib.tfstat_marginalise_static.argtypes = [vp, vp, i32, i32, vp, vp]
    lib.tfstat_plan_info.argtypes = [C.c_int, i32, i32] + grid + [op, C.POINTER(_Plan)]
    lib.tfstat_validate_timestamps.argtypes = [vp, i32, vp, vp, op]
    lib.tfstat_search.argtypes = [vp, i64, i64, vp, i32, i32, C.c_int] + grid + [
        vp, vp, vp, vp, sz, vp, op]
    lib.tfstat_count_terms.argtypes = [vp, i32, C.c_int] + grid + [vp, vp, sz, vp, op]
    lib.tfstat_search_host.argtypes = [vp, i64, i64, vp, i32, i32, C.c_int] + grid + [
        vp, vp, vp, sz, op]
    lib.tfstat_search_host_scratch_bytes.restype = sz
    lib.tfstat_search_host_scratch_bytes.argtypes = [i64, i32, i32, C.c_int] + grid + [C.c_int, op]
    lib.tfstat_general_workspace_bytes.restype = sz
    lib.tfstat_general_workspace_bytes.argtypes = [i32, i32]
    lib.tfstat_map_general.argtypes = [vp, i64, vp, i32, C.POINTER(_Window), vp, i32, vp, i32,
                                       vp, vp, vp, vp, sz, vp, op]
    lib.tfstat_merge_detectors.argtypes = [vp, vp, vp, vp, vp, i32, i32, vp, i32, vp, i64, i64, vp,
                                           op]
    _lib = lib
    return lib


def load_probe_library():
    """dlopen libtfstat_probe.so, the bench-only ALU micro-benchmarks (include/tfstat_probe.h)."""
    global _probe_lib
    if _probe_lib is not None:
        return _probe_lib
    if not os.path.exists(_PROBE_LIB_PATH):
        raise TfstatError(f"{_PROBE_LIB_PATH} is missing: `python -m paper_1805_05652_b200.build`")
    lib = C.CDLL(_PROBE_LIB_PATH)
    lib.tfstat_probe_alu.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double),
                                     C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.tfstat_probe_direct_loop.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double),
                                             C.POINTER(C.c_double)]
    _probe_lib = lib
    return lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        lib = load_library()
        msg = lib.tfstat_strerror(rc).decode()
        extra = f" (cudaError {lib.tfstat_last_cuda_error()})" if rc == -3 else ""
        raise TfstatError(f"{what}: {msg}{extra} [status {rc}]")


def _grid_args(g):
    return [int(g.t0_min), int(g.dt0), int(g.N_t0), int(g.tau_min), int(g.dtau), int(g.N_tau)]


def _opts(min_atoms: int, exp_method: int, events=None, tile=None, rect_method: int = 0,
          stats: Optional[torch.Tensor] = None) -> _Opts:
    o = _Opts()
    if stats is not None:  # CUDA int64 tensor of N_STATS counters the kernels add to
        if not (stats.is_cuda and stats.dtype == torch.int64 and stats.numel() >= N_STATS
                and stats.is_contiguous()):
            raise TfstatError("stats must be a contiguous CUDA int64 tensor of N_STATS entries")
        o.stats = stats.data_ptr()
    o.min_atoms = int(min_atoms)
    o.exp_method = int(exp_method)
    o.rect_method = int(rect_method)
    if tile is not None:  # (cells per thread, threads per CTA[, t0 steps per segment]): tuning
        o.tile_c, o.tile_nt = int(tile[0]), int(tile[1])
        if len(tile) > 2:
            o.seg_len = int(tile[2])
    if events is not None:  # (begin, end): recorded torch.cuda.Event(enable_timing=True)
        o.ev_main_begin = int(events[0].cuda_event)
        o.ev_main_end = int(events[1].cuda_event)
    return o


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _dev_f32(x: torch.Tensor, name: str) -> torch.Tensor:
    if not (isinstance(x, torch.Tensor) and x.is_cuda and x.dtype == torch.float32):
        raise TfstatError(f"{name} must be a CUDA float32 tensor")
    return x


def _dev_i32(x: torch.Tensor, name: str) -> torch.Tensor:
    if not (isinstance(x, torch.Tensor) and x.is_cuda and x.dtype == torch.int32
            and x.is_contiguous()):
        raise TfstatError(f"{name} must be a contiguous CUDA int32 tensor")
    return x


def workspace_bytes(window: int, n_atoms: int, n_templates: int, grid, *, min_atoms: int = 2,
                    exp_method: int = EXP_AUTO, tile=None, rect_method: int = 0) -> int:
    lib = load_library()
    o = _opts(min_atoms, exp_method, tile=tile, rect_method=rect_method)
    n = lib.tfstat_workspace_bytes(window, n_atoms, n_templates, *_grid_args(grid), C.byref(o))
    if n == 0:
        raise TfstatError("tfstat_workspace_bytes: invalid problem shape")
    return int(n)


def plan_info(window: int, n_atoms: int, n_templates: int, grid, *, min_atoms: int = 2,
              exp_method: int = EXP_AUTO, tile=None, rect_method: int = 0) -> dict:
    """What the library will run for this problem shape (tfstat_plan_info): the dominant kernel,
    its tile, its CTAs, the launches of one search and the workspace."""
    lib = load_library()
    o = _opts(min_atoms, exp_method, tile=tile, rect_method=rect_method)
    p = _Plan()
    p.struct_size = C.sizeof(_Plan)
    rc = lib.tfstat_plan_info(window, n_atoms, n_templates, *_grid_args(grid), C.byref(o),
                              C.byref(p))
    _check(rc, "tfstat_plan_info")
    d = {k: int(getattr(p, k)) for k, _ in _Plan._fields_ if k != "struct_size"}
    d["kernel_name"] = KERNEL_NAMES.get(d["kernel"], "?")
    return d


def validate_timestamps(t_atoms: torch.Tensor, *, stream=None) -> int:
    """Opt-in check of the precondition: index of the first time stamp that is not greater than
    its predecessor, or -1 if t_atoms is strictly increasing (tfstat_validate_timestamps)."""
    lib = load_library()
    _dev_i32(t_atoms, "t_atoms")
    out = torch.empty(1, dtype=torch.int32, device=t_atoms.device)
    rc = lib.tfstat_validate_timestamps(t_atoms.data_ptr(), int(t_atoms.shape[0]), out.data_ptr(),
                                        _stream_ptr(stream), None)
    _check(rc, "tfstat_validate_timestamps")
    return int(out.item())


def _workspace(nbytes: int, device, workspace: Optional[torch.Tensor]) -> torch.Tensor:
    if workspace is not None:
        if workspace.numel() * workspace.element_size() < nbytes:
            raise TfstatError("workspace tensor too small")
        return workspace
    return torch.empty(nbytes, dtype=torch.uint8, device=device)


@dataclass
class Results:
    """Marginals of T maps; `raw` is the [T,5] int32 device image of tfstat_result[T]."""

    raw: torch.Tensor
    maps: Optional[torch.Tensor] = None
    flags: Optional[torch.Tensor] = None

    def numpy(self) -> np.ndarray:
        return self.raw.cpu().numpy().view(RESULT_DTYPE).reshape(-1)

    @property
    def max2F(self) -> torch.Tensor:
        return self.raw[:, 0].view(torch.float32)

    @property
    def logB(self) -> torch.Tensor:
        return self.raw[:, 3].view(torch.float32)


def tfstat_map(atoms: torch.Tensor, t_atoms: torch.Tensor, window: int, grid, *,
               min_atoms: int = 2, exp_method: int = EXP_AUTO, want_flags: bool = False,
               out_map: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None,
               stream=None, tile=None, rect_method: int = 0):
    """atoms [7, N] (row stride = ld) -> (map [N_t0, N_tau] fp32 of 2F, flags uint8 or None)."""
    lib = load_library()
    _dev_f32(atoms, "atoms")
    _dev_i32(t_atoms, "t_atoms")
    if atoms.dim() != 2 or atoms.shape[0] != 7 or atoms.stride(1) != 1:
        raise TfstatError("atoms must be [7, N] with unit stride along N")
    n_atoms, ld = int(t_atoms.shape[0]), int(atoms.stride(0))
    if atoms.shape[1] != n_atoms:
        raise TfstatError("atoms / t_atoms length mismatch")
    dev = atoms.device
    if out_map is None:
        out_map = torch.empty((grid.N_t0, grid.N_tau), dtype=torch.float32, device=dev)
    flags = (torch.empty((grid.N_t0, grid.N_tau), dtype=torch.uint8, device=dev)
             if want_flags else None)
    nbytes = workspace_bytes(window, n_atoms, 1, grid, min_atoms=min_atoms, exp_method=exp_method,
                             tile=tile, rect_method=rect_method)
    ws = _workspace(nbytes, dev, workspace)
    o = _opts(min_atoms, exp_method, tile=tile, rect_method=rect_method)
    rc = lib.tfstat_map(atoms.data_ptr(), ld, t_atoms.data_ptr(), n_atoms, window,
                        *_grid_args(grid), out_map.data_ptr(),
                        flags.data_ptr() if flags is not None else None, ws.data_ptr(), nbytes,
                        _stream_ptr(stream), C.byref(o))
    _check(rc, "tfstat_map")
    return out_map, flags


def tfstat_marginalise(map2F: torch.Tensor, flags: Optional[torch.Tensor] = None, *,
                       stream=None) -> Results:
    lib = load_library()
    _dev_f32(map2F, "map")
    if map2F.dim() != 2 or not map2F.is_contiguous():
        raise TfstatError("map must be a contiguous [N_t0, N_tau] tensor")
    if flags is not None and not (flags.is_cuda and flags.dtype == torch.uint8
                                  and flags.is_contiguous() and flags.shape == map2F.shape):
        raise TfstatError("flags must be a contiguous CUDA uint8 tensor shaped like map")
    N_t0, N_tau = map2F.shape
    nbytes = int(lib.tfstat_marginalise_workspace_bytes(N_t0, N_tau))
    ws = torch.empty(nbytes, dtype=torch.uint8, device=map2F.device)
    out = torch.empty((1, 5), dtype=torch.int32, device=map2F.device)
    rc = lib.tfstat_marginalise(map2F.data_ptr(), flags.data_ptr() if flags is not None else None,
                                N_t0, N_tau, out.data_ptr(), ws.data_ptr(), nbytes,
                                _stream_ptr(stream), None)
    _check(rc, "tfstat_marginalise")
    return Results(out)


def tfstat_marginalise_static(map2F: torch.Tensor, flags: Optional[torch.Tensor] = None, *,
                              out: Optional[torch.Tensor] = None, stream=None) -> Results:
    """tfstat_marginalise without a workspace: the library's static device scratch is used and
    nothing is allocated by the call (pass `out`, a [1, 5] int32 CUDA tensor, to keep torch from
    allocating either).  Calls that overlap on the GPU race on the scratch (include/tfstat.h)."""
    lib = load_library()
    _dev_f32(map2F, "map")
    if map2F.dim() != 2 or not map2F.is_contiguous():
        raise TfstatError("map must be a contiguous [N_t0, N_tau] tensor")
    if flags is not None and not (flags.is_cuda and flags.dtype == torch.uint8
                                  and flags.is_contiguous() and flags.shape == map2F.shape):
        raise TfstatError("flags must be a contiguous CUDA uint8 tensor shaped like map")
    N_t0, N_tau = map2F.shape
    if out is None:
        out = torch.empty((1, 5), dtype=torch.int32, device=map2F.device)
    elif not (out.is_cuda and out.dtype == torch.int32 and out.is_contiguous()
              and out.numel() == 5):
        raise TfstatError("out must be a contiguous CUDA int32 tensor of 5 elements")
    with torch.cuda.device(map2F.device):  # the static scratch is looked up on the CURRENT device
        rc = lib.tfstat_marginalise_static(map2F.data_ptr(),
                                           flags.data_ptr() if flags is not None else None,
                                           N_t0, N_tau, out.data_ptr(), _stream_ptr(stream))
    _check(rc, "tfstat_marginalise_static")
    return Results(out.view(1, 5))


def tfstat_search(atoms: torch.Tensor, t_atoms: torch.Tensor, window: int, grid, *,
                  min_atoms: int = 2, exp_method: int = EXP_AUTO, want_maps: bool = False,
                  want_flags: bool = False, workspace: Optional[torch.Tensor] = None,
                  out: Optional[torch.Tensor] = None, stream=None,
                  main_kernel_events=None, tile=None, rect_method: int = 0,
                  stats: Optional[torch.Tensor] = None) -> Results:
    """atoms [T, 7, N] -> marginals of the T maps (and the maps / flags if asked)."""
    lib = load_library()
    _dev_f32(atoms, "atoms")
    _dev_i32(t_atoms, "t_atoms")
    if atoms.dim() != 3 or atoms.shape[1] != 7 or atoms.stride(2) != 1:
        raise TfstatError("atoms must be [T, 7, N] with unit stride along N")
    T, n_atoms = int(atoms.shape[0]), int(t_atoms.shape[0])
    if atoms.shape[2] != n_atoms:
        raise TfstatError("atoms / t_atoms length mismatch")
    tstride, ld = int(atoms.stride(0)), int(atoms.stride(1))
    dev = atoms.device
    if out is None:
        out = torch.empty((T, 5), dtype=torch.int32, device=dev)
    maps = (torch.empty((T, grid.N_t0, grid.N_tau), dtype=torch.float32, device=dev)
            if want_maps else None)
    flags = (torch.empty((T, grid.N_t0, grid.N_tau), dtype=torch.uint8, device=dev)
             if want_flags else None)
    nbytes = workspace_bytes(window, n_atoms, T, grid, min_atoms=min_atoms, exp_method=exp_method,
                             tile=tile, rect_method=rect_method)
    ws = _workspace(nbytes, dev, workspace)
    o = _opts(min_atoms, exp_method, main_kernel_events, tile=tile, rect_method=rect_method,
              stats=stats)
    rc = lib.tfstat_search(atoms.data_ptr(), tstride, ld, t_atoms.data_ptr(), n_atoms, T, window,
                           *_grid_args(grid), out.data_ptr(),
                           maps.data_ptr() if maps is not None else None,
                           flags.data_ptr() if flags is not None else None, ws.data_ptr(), nbytes,
                           _stream_ptr(stream), C.byref(o))
    _check(rc, "tfstat_search")
    return Results(out, maps, flags)


def tfstat_map_general(atoms: torch.Tensor, t_atoms: torch.Tensor, kind: int, support,
                       t0_grid: torch.Tensor, tau_grid: torch.Tensor, *,
                       table: Optional[torch.Tensor] = None, min_atoms: int = 2,
                       want_map: bool = True, want_flags: bool = False,
                       want_marginals: bool = True, stream=None, cells_per_thread: int = 0):
    """General window on explicit grids (include/tfstat.h, tfstat_map_general).

    atoms [7, N]; t0_grid [N_t0], tau_grid [N_tau]: CUDA int32 tensors of seconds (any order);
    support = (num, den) in units of tau; table: CUDA float32 samples of w(u) for kind TABLE.
    Returns (map or None, flags or None, Results or None)."""
    lib = load_library()
    _dev_f32(atoms, "atoms")
    _dev_i32(t_atoms, "t_atoms")
    _dev_i32(t0_grid, "t0_grid")
    _dev_i32(tau_grid, "tau_grid")
    if atoms.dim() != 2 or atoms.shape[0] != 7 or atoms.stride(1) != 1:
        raise TfstatError("atoms must be [7, N] with unit stride along N")
    n_atoms, ld = int(t_atoms.shape[0]), int(atoms.stride(0))
    if atoms.shape[1] != n_atoms:
        raise TfstatError("atoms / t_atoms length mismatch")
    if not (want_map or want_marginals):
        raise TfstatError("nothing to compute: want_map or want_marginals")
    w = _Window()
    w.kind, w.support_num, w.support_den = int(kind), int(support[0]), int(support[1])
    if table is not None:
        _dev_f32(table, "table")
        if not table.is_contiguous():
            raise TfstatError("table must be contiguous")
        w.n_table, w.table = int(table.numel()), table.data_ptr()
    N_t0, N_tau = int(t0_grid.shape[0]), int(tau_grid.shape[0])
    dev = atoms.device
    out_map = torch.empty((N_t0, N_tau), dtype=torch.float32, device=dev) if want_map else None
    flags = torch.empty((N_t0, N_tau), dtype=torch.uint8, device=dev) if want_flags else None
    out = torch.empty((1, 5), dtype=torch.int32, device=dev) if want_marginals else None
    nbytes = int(lib.tfstat_general_workspace_bytes(N_t0, N_tau))
    ws = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=dev)
    o = _opts(min_atoms, EXP_AUTO)
    o.tile_c = int(cells_per_thread)
    rc = lib.tfstat_map_general(atoms.data_ptr(), ld, t_atoms.data_ptr(), n_atoms, C.byref(w),
                                t0_grid.data_ptr(), N_t0, tau_grid.data_ptr(), N_tau,
                                out_map.data_ptr() if want_map else None,
                                flags.data_ptr() if want_flags else None,
                                out.data_ptr() if want_marginals else None, ws.data_ptr(),
                                ws.numel(), _stream_ptr(stream), C.byref(o))
    _check(rc, "tfstat_map_general")
    return out_map, flags, (Results(out) if want_marginals else None)


def tfstat_merge_detectors(atoms_dets, t_dets, t_out: torch.Tensor, *, stream=None) -> torch.Tensor:
    """Per-detector atoms -> atoms merged per time stamp (include/tfstat.h).

    atoms_dets: list of CUDA float32 tensors [T, 7, N_x] (or [7, N_x]); t_dets: list of CUDA int32
    [N_x]; t_out: CUDA int32 [N] (normally the sorted union).  Returns [T, 7, N] (or [7, N])."""
    lib = load_library()
    n_det = len(atoms_dets)
    if n_det != len(t_dets) or n_det < 1:
        raise TfstatError("need one time-stamp tensor per detector")
    squeeze = atoms_dets[0].dim() == 2
    A = [a[None] if squeeze else a for a in atoms_dets]
    T = int(A[0].shape[0])
    for a, t in zip(A, t_dets):
        _dev_f32(a, "atoms_dets[x]")
        _dev_i32(t, "t_dets[x]")
        if a.dim() != 3 or a.shape[0] != T or a.shape[1] != 7 or a.stride(2) != 1 \
                or a.shape[2] != t.shape[0]:
            raise TfstatError("atoms_dets[x] must be [T, 7, N_x] matching t_dets[x]")
    _dev_i32(t_out, "t_out")
    n_out = int(t_out.shape[0])
    out = torch.empty((T, 7, n_out), dtype=torch.float32, device=t_out.device)
    pa = (C.c_void_p * n_det)(*[a.data_ptr() for a in A])
    pt = (C.c_void_p * n_det)(*[t.data_ptr() for t in t_dets])
    ts = (C.c_int64 * n_det)(*[int(a.stride(0)) for a in A])
    lds = (C.c_int64 * n_det)(*[int(a.stride(1)) for a in A])
    ns = (C.c_int32 * n_det)(*[int(t.shape[0]) for t in t_dets])
    rc = lib.tfstat_merge_detectors(pa, ts, lds, pt, ns, n_det, T, t_out.data_ptr(), n_out,
                                    out.data_ptr(), 7 * n_out, n_out, _stream_ptr(stream), None)
    _check(rc, "tfstat_merge_detectors")
    return out[0] if squeeze else out


def count_terms(t_atoms: torch.Tensor, window: int, grid, *, stream=None) -> int:
    """N_sums of eqs. (A.5)/(A.6) with gaps: total (cell, atom-in-window) pairs of the grid."""
    lib = load_library()
    _dev_i32(t_atoms, "t_atoms")
    n_atoms = int(t_atoms.shape[0])
    nbytes = workspace_bytes(window, n_atoms, 1, grid)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=t_atoms.device)
    out = torch.zeros(1, dtype=torch.int64, device=t_atoms.device)
    rc = lib.tfstat_count_terms(t_atoms.data_ptr(), n_atoms, window, *_grid_args(grid),
                                out.data_ptr(), ws.data_ptr(), nbytes, _stream_ptr(stream), None)
    _check(rc, "tfstat_count_terms")
    return int(out.item())


_host_scratch: Optional[torch.Tensor] = None  # device scratch reused by tfstat_search_host


def search_host_scratch_bytes(template_stride: int, n_atoms: int, n_templates: int, window: int,
                              grid, *, want_maps: bool = False, min_atoms: int = 2,
                              exp_method: int = EXP_AUTO) -> int:
    """Device scratch tfstat_search_host wants for chunks of min(n_templates, 256) templates."""
    lib = load_library()
    o = _opts(min_atoms, exp_method)
    n = int(lib.tfstat_search_host_scratch_bytes(int(template_stride), n_atoms, n_templates,
                                                 window, *_grid_args(grid), int(want_maps),
                                                 C.byref(o)))
    if n == 0:
        raise TfstatError("tfstat_search_host_scratch_bytes: invalid problem shape")
    return n


def tfstat_search_host(atoms: torch.Tensor, t_atoms: torch.Tensor, window: int, grid, *,
                       min_atoms: int = 2, exp_method: int = EXP_AUTO, want_maps: bool = False,
                       max_device_bytes: int = 0, scratch: Optional[torch.Tensor] = None,
                       library_malloc: bool = False):
    """End-to-end call on HOST tensors (pinned for overlap): H2D copies, fused search and D2H
    of the results all happen inside the library.  Returns (results ndarray, maps or None).

    The device scratch buffer is a torch tensor kept between calls (or `scratch`, a CUDA uint8
    tensor of the caller); `max_device_bytes` > 0 caps its size (smaller chunks);
    `library_malloc` passes no scratch at all: the library cudaMallocs and frees its own."""
    global _host_scratch
    lib = load_library()
    if atoms.is_cuda or t_atoms.is_cuda:
        raise TfstatError("tfstat_search_host takes host (CPU) tensors")
    if atoms.dtype != torch.float32 or t_atoms.dtype != torch.int32:
        raise TfstatError("atoms must be float32 and t_atoms int32")
    if atoms.dim() != 3 or atoms.shape[1] != 7 or atoms.stride(2) != 1:
        raise TfstatError("atoms must be [T, 7, N] with unit stride along N")
    T, n_atoms = int(atoms.shape[0]), int(t_atoms.shape[0])
    out = torch.empty((T, 5), dtype=torch.int32).pin_memory()
    maps = (torch.empty((T, grid.N_t0, grid.N_tau), dtype=torch.float32).pin_memory()
            if want_maps else None)
    o = _opts(min_atoms, exp_method)
    # The library works on streams of its own and returns when everything has completed.  A torch
    # scratch tensor may be a block the caching allocator has just taken back from work that is
    # still running on the current stream (e.g. the workspace of an earlier tfstat_search):
    # stream-ordered reuse is only safe on that stream, so let it drain first.
    torch.cuda.current_stream().synchronize()
    if library_malloc:
        rc = lib.tfstat_search_host(atoms.data_ptr(), int(atoms.stride(0)), int(atoms.stride(1)),
                                    t_atoms.data_ptr(), n_atoms, T, window, *_grid_args(grid),
                                    out.data_ptr(),
                                    maps.data_ptr() if maps is not None else None, None,
                                    int(max_device_bytes), C.byref(o))
        _check(rc, "tfstat_search_host")
        return out.numpy().view(RESULT_DTYPE).reshape(-1), maps
    if scratch is None:
        need = int(lib.tfstat_search_host_scratch_bytes(int(atoms.stride(0)), n_atoms, T, window,
                                                        *_grid_args(grid), int(want_maps),
                                                        C.byref(o)))
        if need == 0:
            raise TfstatError("tfstat_search_host_scratch_bytes: invalid problem shape")
        if max_device_bytes:
            need = min(need, int(max_device_bytes))
        if _host_scratch is None or _host_scratch.numel() < need:
            _host_scratch = None
            _host_scratch = torch.empty(need, dtype=torch.uint8, device="cuda")
        scratch, nbytes = _host_scratch, need
    else:
        if not (scratch.is_cuda and scratch.dtype == torch.uint8 and scratch.is_contiguous()):
            raise TfstatError("scratch must be a contiguous CUDA uint8 tensor")
        nbytes = scratch.numel()
    rc = lib.tfstat_search_host(atoms.data_ptr(), int(atoms.stride(0)), int(atoms.stride(1)),
                                t_atoms.data_ptr(), n_atoms, T, window, *_grid_args(grid),
                                out.data_ptr(), maps.data_ptr() if maps is not None else None,
                                scratch.data_ptr(), nbytes, C.byref(o))
    _check(rc, "tfstat_search_host")
    return out.numpy().view(RESULT_DTYPE).reshape(-1), maps


PROBE_KINDS = {"ffma": 0, "fadd": 1, "mufu_ex2": 2, "ffma2": 3, "fadd2": 4, "ffma_mufu": 5,
               "lds128": 6, "dfma": 7,
               "ffma2_two_pairs": 8, "ffma2_scalar_pair": 9, "ffma2_two_scalars": 10}


def probe_alu(kind: str, reps: int = 3) -> dict:
    """Measured issue rate of one instruction class on the current GPU (tfstat_probe.h; the
    bench-only libtfstat_probe.so)."""
    lib = load_probe_library()
    a, b, c = C.c_double(0), C.c_double(0), C.c_double(0)
    rc = lib.tfstat_probe_alu(PROBE_KINDS[kind], reps, C.byref(a), C.byref(b), C.byref(c))
    if rc != 0:
        raise TfstatError(f"tfstat_probe_alu({kind}): status {rc}")
    return dict(kind=kind, lane_ops_per_s=a.value, ops_per_clk_sm=b.value, sm_mhz=c.value)


def probe_direct_loop(form: int, cells: int, reps: int = 200) -> dict:
    """The isolated core loop of the direct exponential sum in one of its two accumulator layouts
    (tfstat_probe.h): 0 = channel pairs (scalar x register pair), 1 = cell pairs (two scalars);
    2, 3 = cell pairs with two / four more LDS.128 per atom whose results are not used."""
    lib = load_probe_library()
    a, b = C.c_double(0), C.c_double(0)
    rc = lib.tfstat_probe_direct_loop(int(form), int(cells), int(reps), C.byref(a), C.byref(b))
    if rc != 0:
        raise TfstatError(f"tfstat_probe_direct_loop({form}, {cells}): status {rc}")
    names = ("channel_pairs", "cell_pairs", "cell_pairs_plus_2_lds128", "cell_pairs_plus_4_lds128")
    return dict(form=names[form], cells=cells,
                terms_per_clk_sm=a.value, terms_per_s=b.value)
