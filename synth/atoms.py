"""Synthetic atom sets (BASELINE.json `configs`; SURVEY.md section 8(d) recipe).

Stand-in for the PyFstat-simulated data of the paper.
Everything is computed in fp64 and stored as fp32, like the paper's real32
atoms.

Atom model (BASELINE.json configs[0]):
    detectors d in {0,1}, sidereal period 86164 s, per-template phase phi
      a_d(t) = 0.4 cos(2 pi t/86164 + 0.3 + d + phi) + 0.2
      b_d(t) = 0.35 sin(2 pi t/86164 + 1.1 + d + phi) - 0.1
      a2 = sum_d a_d^2,  b2 = sum_d b_d^2,  ab = sum_d a_d b_d
    noise n_d complex with Re, Im ~ N(0, 1/2):
      Fa = sum_d a_d n_d,  Fb = sum_d b_d n_d
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np

TSFT = 1800  # s
SIDEREAL_DAY = 86164.0  # s
BASE_SEED = 180505652 * 10  # + config id


@dataclass
class Grid:
    """Uniform (t0, tau) grid, integer seconds."""

    t0_min: int
    dt0: int
    N_t0: int
    tau_min: int
    dtau: int
    N_tau: int

    @property
    def n_cells(self) -> int:
        return self.N_t0 * self.N_tau

    def t0(self) -> np.ndarray:
        return self.t0_min + self.dt0 * np.arange(self.N_t0, dtype=np.int64)

    def tau(self) -> np.ndarray:
        return self.tau_min + self.dtau * np.arange(self.N_tau, dtype=np.int64)


@dataclass
class AtomSet:
    """`atoms`: [T, 7, N] fp32, rows a2,b2,ab,FaRe,FaIm,FbRe,FbIm.
    `t`: [N] int32 start times, strictly increasing, shared by all T templates."""

    atoms: np.ndarray
    t: np.ndarray

    @property
    def n_templates(self) -> int:
        return self.atoms.shape[0]

    @property
    def n_atoms(self) -> int:
        return self.atoms.shape[2]


def template_seed(config_id: int, template: int = 0) -> np.random.SeedSequence:
    """SeedSequence for one template of one config (spawn-key = template)."""
    return np.random.SeedSequence(BASE_SEED + config_id, spawn_key=(template,))


def antenna_terms(t: np.ndarray, phi: float = 0.0) -> Tuple[np.ndarray, np.ndarray]:
    """a_d(t), b_d(t) for d in {0,1}; returns arrays of shape [2, N] (fp64)."""
    t = np.asarray(t, dtype=np.float64)
    d = np.arange(2, dtype=np.float64)[:, None]
    arg = 2.0 * np.pi * t[None, :] / SIDEREAL_DAY
    a = 0.4 * np.cos(arg + 0.3 + d + phi) + 0.2
    b = 0.35 * np.sin(arg + 1.1 + d + phi) - 0.1
    return a, b


def gap_mask(n_slots: int, frac: float, rng: np.random.Generator,
             mean_len: float = 24.0) -> np.ndarray:
    """Boolean keep-mask over SFT slots with exactly round(frac*n_slots) removed.

    Contiguous runs of length 1+Geometric(mean `mean_len`) are removed at uniform
    random starts until the quota is met (the last run is trimmed to hit it)."""
    keep = np.ones(n_slots, dtype=bool)
    quota = int(round(frac * n_slots))
    removed = 0
    p = 1.0 / mean_len
    while removed < quota:
        length = 1 + int(rng.geometric(p))
        start = int(rng.integers(0, n_slots))
        for s in range(start, min(start + length, n_slots)):
            if removed >= quota:
                break
            if keep[s]:
                keep[s] = False
                removed += 1
    return keep


def make_atoms(t: np.ndarray, rng: np.random.Generator, phi: float = 0.0,
               noise: bool = True) -> np.ndarray:
    """One template's atoms, [7, N] fp64 (caller rounds to fp32)."""
    a, b = antenna_terms(t, phi)
    n = t.shape[0]
    out = np.empty((7, n), dtype=np.float64)
    out[0] = (a * a).sum(0)
    out[1] = (b * b).sum(0)
    out[2] = (a * b).sum(0)
    if noise:
        z = rng.normal(0.0, np.sqrt(0.5), size=(2, 2, n))  # [d, re/im, N]
        nd = z[:, 0, :] + 1j * z[:, 1, :]
    else:
        nd = np.zeros((2, n), dtype=np.complex128)
    fa = (a * nd).sum(0)
    fb = (b * nd).sum(0)
    out[3], out[4] = fa.real, fa.imag
    out[5], out[6] = fb.real, fb.imag
    return out


def make_detector_atoms(t: np.ndarray, rng: np.random.Generator, phi: float = 0.0) -> np.ndarray:
    """The same atom model per detector, NOT merged: [2, 7, N] fp64 with rows a_d^2, b_d^2,
    a_d b_d, Re/Im(a_d n_d), Re/Im(b_d n_d).  Draws the noise exactly like `make_atoms`, so for
    the same generator state the sum over d is `make_atoms` up to fp64 rounding order.  Input
    for the per-detector entry point (tfstat_merge_detectors): each detector may then keep its
    own subset of the time stamps."""
    a, b = antenna_terms(t, phi)
    n = t.shape[0]
    z = rng.normal(0.0, np.sqrt(0.5), size=(2, 2, n))  # [d, re/im, N]
    nd = z[:, 0, :] + 1j * z[:, 1, :]
    out = np.empty((2, 7, n), dtype=np.float64)
    out[:, 0], out[:, 1], out[:, 2] = a * a, b * b, a * b
    fa, fb = a * nd, b * nd
    out[:, 3], out[:, 4] = fa.real, fa.imag
    out[:, 5], out[:, 6] = fb.real, fb.imag
    return out


def _inject(atoms32: np.ndarray, W: np.ndarray, rho: float,
            rng: np.random.Generator) -> Tuple[complex, complex]:
    """Add W*(c1 a2 + c2 ab) to Fa and W*(c1 ab + c2 b2) to Fb in place.

    c1, c2 ~ complex N(0,1), rescaled so that 2(A|c1|^2 + B|c2|^2 + 2C Re(c1 c2*))
    equals rho^2 with A,B,C the W^2-weighted sums."""
    a2 = atoms32[0].astype(np.float64)
    b2 = atoms32[1].astype(np.float64)
    ab = atoms32[2].astype(np.float64)
    c = rng.normal(size=4)
    c1, c2 = complex(c[0], c[1]), complex(c[2], c[3])
    W2 = W * W
    A, B, C = (W2 * a2).sum(), (W2 * b2).sum(), (W2 * ab).sum()
    rho2_raw = 2.0 * (A * abs(c1) ** 2 + B * abs(c2) ** 2
                      + 2.0 * C * (c1 * np.conj(c2)).real)
    s = rho / np.sqrt(rho2_raw)
    c1, c2 = c1 * s, c2 * s
    fa = W * (c1 * a2 + c2 * ab)
    fb = W * (c1 * ab + c2 * b2)
    f64 = atoms32.astype(np.float64)
    f64[3] += fa.real
    f64[4] += fa.imag
    f64[5] += fb.real
    f64[6] += fb.imag
    atoms32[3:7] = f64[3:7].astype(np.float32)
    return c1, c2


def inject_exponential(atoms32: np.ndarray, t: np.ndarray, t0_sig: int,
                       tau_sig: int, rho: float,
                       rng: np.random.Generator) -> Tuple[complex, complex]:
    """Exponential-window injection, half-open 3 tau cut (BASELINE.json configs[1])."""
    dt = t.astype(np.float64) - float(t0_sig)
    inside = (t >= t0_sig) & (t < t0_sig + 3 * tau_sig)
    W = np.where(inside, np.exp(-np.where(inside, dt, 0.0) / float(tau_sig)), 0.0)
    return _inject(atoms32, W, rho, rng)


def inject_rectangular(atoms32: np.ndarray, t: np.ndarray, t0_sig: int,
                       tau_sig: int, rho: float,
                       rng: np.random.Generator) -> Tuple[complex, complex]:
    inside = (t >= t0_sig) & (t < t0_sig + tau_sig)
    return _inject(atoms32, inside.astype(np.float64), rho, rng)


def pack_atoms(per_template: list) -> np.ndarray:
    """Stack per-template [7,N] arrays into the [T,7,N] fp32 layout."""
    return np.ascontiguousarray(np.stack(per_template).astype(np.float32))
