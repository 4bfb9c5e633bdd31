"""ctypes marshalling for oracle/tfstat_oracle.c (no arithmetic here)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np

RECT, EXP, TABLE = 0, 1, 2
_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tfstat_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_tfstat.so")
_lib = None


class _Result(C.Structure):
    _fields_ = [("max2F", C.c_double), ("m", C.c_int32), ("n", C.c_int32),
                ("logB", C.c_double), ("n_valid", C.c_int32), ("pad_", C.c_int32)]


@dataclass
class OracleResult:
    max2F: float
    m: int
    n: int
    logB: float
    n_valid: int


def build(force: bool = False) -> str:
    """gcc -O2 (no fast-math) -fopenmp -> oracle/liboracle_tfstat.so."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + f".tmp{os.getpid()}"
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-Wall", "-o", tmp,
           _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        i32, i64, vp = C.c_int32, C.c_int64, C.c_void_p
        grid = [i32] * 6
        lib.oracle_tfstat_map.argtypes = [vp, i64, vp, i32, C.c_int] + grid + [
            i32, vp, vp, vp, vp, C.c_int]
        lib.oracle_tfstat_cells.argtypes = [vp, i64, vp, i32, C.c_int] + grid + [
            i32, vp, vp, i64, vp, vp, vp, vp, C.c_int]
        lib.oracle_tfstat_marginalise.argtypes = [vp, vp, i32, i32, C.POINTER(_Result)]
        lib.oracle_tfstat_search.argtypes = [vp, i64, i64, vp, i32, i32, C.c_int] + grid + [
            i32, vp, vp, C.c_int]
        lib.oracle_tfstat_map_general.argtypes = [vp, i64, vp, i32, C.c_int, i32, i32, vp, i32,
                                                  vp, i32, vp, i32, i32, vp, vp, vp, vp, C.c_int]
        lib.oracle_num_threads.restype = C.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _check_atoms(atoms: np.ndarray, t: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    atoms = np.ascontiguousarray(atoms, dtype=np.float32)
    t = np.ascontiguousarray(t, dtype=np.int32)
    assert atoms.ndim == 2 and atoms.shape[0] == 7 and atoms.shape[1] == t.shape[0]
    return atoms, t


def map2F(atoms, t, window, grid, min_atoms: int = 2, n_threads: int = 0):
    """Full map.  Returns dict(twoF[N_t0,N_tau] f64, flags u8, cond f64, cnt i32)."""
    atoms, t = _check_atoms(atoms, t)
    shape = (grid.N_t0, grid.N_tau)
    twoF = np.empty(shape, np.float64)
    flags = np.empty(shape, np.uint8)
    cond = np.empty(shape, np.float64)
    cnt = np.empty(shape, np.int32)
    rc = _load().oracle_tfstat_map(_ptr(atoms), atoms.shape[1], _ptr(t), t.shape[0], window,
                                   grid.t0_min, grid.dt0, grid.N_t0, grid.tau_min, grid.dtau,
                                   grid.N_tau, min_atoms, _ptr(twoF), _ptr(flags), _ptr(cond),
                                   _ptr(cnt), n_threads)
    if rc != 0:
        raise ValueError(f"oracle_tfstat_map rc={rc}")
    return dict(twoF=twoF, flags=flags, cond=cond, cnt=cnt)


def map2F_general(atoms, t, kind, support, t0_grid, tau_grid, table=None, min_atoms: int = 2,
                  n_threads: int = 0):
    """General window on explicit grids.  support = (num, den) in units of tau; table = fp32
    samples of w(u) for kind TABLE.  Returns the same dict as map2F."""
    atoms, t = _check_atoms(atoms, t)
    t0_grid = np.ascontiguousarray(t0_grid, dtype=np.int32)
    tau_grid = np.ascontiguousarray(tau_grid, dtype=np.int32)
    tab = None if table is None else np.ascontiguousarray(table, dtype=np.float32)
    shape = (t0_grid.shape[0], tau_grid.shape[0])
    twoF = np.empty(shape, np.float64)
    flags = np.empty(shape, np.uint8)
    cond = np.empty(shape, np.float64)
    cnt = np.empty(shape, np.int32)
    rc = _load().oracle_tfstat_map_general(
        _ptr(atoms), atoms.shape[1], _ptr(t), t.shape[0], kind, int(support[0]), int(support[1]),
        _ptr(tab), 0 if tab is None else tab.shape[0], _ptr(t0_grid), shape[0], _ptr(tau_grid),
        shape[1], min_atoms, _ptr(twoF), _ptr(flags), _ptr(cond), _ptr(cnt), n_threads)
    if rc != 0:
        raise ValueError(f"oracle_tfstat_map_general rc={rc}")
    return dict(twoF=twoF, flags=flags, cond=cond, cnt=cnt)


def merge_detectors(atoms_dets, t_dets, t_out):
    """atoms_dets: list of [7, N_x] fp32 arrays, t_dets: list of [N_x] int32 -> [7, len(t_out)] fp32."""
    n_det = len(atoms_dets)
    A = [np.ascontiguousarray(a, dtype=np.float32) for a in atoms_dets]
    T = [np.ascontiguousarray(t, dtype=np.int32) for t in t_dets]
    t_out = np.ascontiguousarray(t_out, dtype=np.int32)
    out = np.empty((7, t_out.shape[0]), np.float32)
    pa = (C.c_void_p * n_det)(*[a.ctypes.data for a in A])
    pt = (C.c_void_p * n_det)(*[t.ctypes.data for t in T])
    lds = (C.c_int64 * n_det)(*[a.shape[1] for a in A])
    ns = (C.c_int32 * n_det)(*[t.shape[0] for t in T])
    lib = _load()
    lib.oracle_merge_detectors.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                           C.c_int32, C.c_void_p, C.c_int32, C.c_void_p,
                                           C.c_int64]
    rc = lib.oracle_merge_detectors(pa, lds, pt, ns, n_det, _ptr(t_out), t_out.shape[0],
                                    _ptr(out), out.shape[1])
    if rc != 0:
        raise ValueError(f"oracle_merge_detectors rc={rc}")
    return out


def cells(atoms, t, window, grid, ms, ns, min_atoms: int = 2, n_threads: int = 0):
    """The same per-cell definition on a list of (m, n) cells."""
    atoms, t = _check_atoms(atoms, t)
    ms = np.ascontiguousarray(ms, dtype=np.int32)
    ns = np.ascontiguousarray(ns, dtype=np.int32)
    K = ms.shape[0]
    twoF = np.empty(K, np.float64)
    flags = np.empty(K, np.uint8)
    cond = np.empty(K, np.float64)
    cnt = np.empty(K, np.int32)
    rc = _load().oracle_tfstat_cells(_ptr(atoms), atoms.shape[1], _ptr(t), t.shape[0], window,
                                     grid.t0_min, grid.dt0, grid.N_t0, grid.tau_min,
                                     grid.dtau, grid.N_tau, min_atoms, _ptr(ms), _ptr(ns), K,
                                     _ptr(twoF), _ptr(flags), _ptr(cond), _ptr(cnt), n_threads)
    if rc != 0:
        raise ValueError(f"oracle_tfstat_cells rc={rc}")
    return dict(twoF=twoF, flags=flags, cond=cond, cnt=cnt)


def marginalise(map2F_, flags=None) -> OracleResult:
    m = np.ascontiguousarray(map2F_, dtype=np.float64)
    assert m.ndim == 2
    f = None if flags is None else np.ascontiguousarray(flags, dtype=np.uint8)
    r = _Result()
    rc = _load().oracle_tfstat_marginalise(_ptr(m), _ptr(f), m.shape[0], m.shape[1], C.byref(r))
    if rc != 0:
        raise ValueError(f"oracle_tfstat_marginalise rc={rc}")
    return OracleResult(r.max2F, r.m, r.n, r.logB, r.n_valid)


def search(atoms, t, window, grid, min_atoms: int = 2, n_threads: int = 0):
    """Batched search over atoms[T,7,N].  Returns (list[OracleResult], n_terms)."""
    atoms = np.ascontiguousarray(atoms, dtype=np.float32)
    t = np.ascontiguousarray(t, dtype=np.int32)
    assert atoms.ndim == 3 and atoms.shape[1] == 7 and atoms.shape[2] == t.shape[0]
    T, _, N = atoms.shape
    res = (_Result * T)()
    terms = C.c_int64(0)
    rc = _load().oracle_tfstat_search(_ptr(atoms), 7 * N, N, _ptr(t), N, T, window,
                                      grid.t0_min, grid.dt0, grid.N_t0, grid.tau_min,
                                      grid.dtau, grid.N_tau, min_atoms,
                                      C.cast(res, C.c_void_p), C.addressof(terms), n_threads)
    if rc != 0:
        raise ValueError(f"oracle_tfstat_search rc={rc}")
    return ([OracleResult(r.max2F, r.m, r.n, r.logB, r.n_valid) for r in res],
            int(terms.value))
