"""Fit the paper's timing model of the F-statistic map function on this GPU (Appendix A).

    python -m paper_1805_05652_b200.timing_model [--out fit.json] [--max-days 365] [--quick]

Model (eqs. A.3, A.4), per single-template map call:

    cost_e = c_call + c_SFTs N_SFT + c_sums^e N_sums^e + c_F N_t0 N_tau
    cost_r = c_call + c_SFTs N_SFT + c_sums^r N_sums^r + c_F N_t0 N_tau

with N_sums from eqs. (A.5)/(A.6), here counted exactly on the device by
tfstat_count_terms.  `c_call` is NOT in the paper: a GPU call is a chain of kernel launches whose
fixed latency would otherwise be booked on c_SFTs; it is fitted together with c_SFTs in step (i).
The fit follows the paper's three steps:
  (i)   c_call + c_SFTs N_SFT on short data sets (N_sums <= 100 in the paper; here: the shortest
        setups of the sweep, cells <= 4096),
  (ii)  with those fixed, c_sums^r N_sums^r + c_F N_t0 N_tau on rectangular-window runs,
  (iii) with c_call, c_SFTs, c_F fixed, c_sums^e N_sums^e on exponential-window runs,
and then the PGM-equivalent constants c_r = c_sums^r + c_F (A.7) and c_e = 3 c_sums^e (A.8,
PAPER.md:245-249) that Table 1 lists for CPUs and pyCUDA GPUs.

Setups are the paper's: gapless data, T_SFT = 1800 s, dt0 = dtau = T_SFT,
t0 in [0, T_data - 2 T_SFT], tau in [2 T_SFT, T_data] ('overlapping' case), plus 'embedded'
ones (t0 in the first half, tau up to a quarter of the data) so that N_sums and N_t0 N_tau do
not scale together.  Only the map function is timed (CUDA events, atoms resident on the
device, full map written), as in the paper's Appendix-A fit.  The least-squares algebra here is
analysis of measured times, not part of the hot path.
"""
from __future__ import annotations

import argparse
import json
import statistics
import sys

import numpy as np
import torch

from . import binding as B

TSFT = 1800


def _atoms(n_atoms: int, seed: int = 1):
    """Gapless two-detector atoms of the seeded input generators (`synth/`: the one
    place the atom model lives; values only matter through the conditioning of the cells)."""
    from synth.atoms import make_atoms  # the repo's input generators, not part of the product

    t = np.arange(n_atoms, dtype=np.int64) * TSFT
    atoms = make_atoms(t, np.random.default_rng(seed)).astype(np.float32)
    return (torch.from_numpy(atoms).cuda().contiguous(),
            torch.from_numpy(t.astype(np.int32)).cuda().contiguous())


class _Grid:
    def __init__(self, t0_min, dt0, N_t0, tau_min, dtau, N_tau):
        self.t0_min, self.dt0, self.N_t0 = t0_min, dt0, N_t0
        self.tau_min, self.dtau, self.N_tau = tau_min, dtau, N_tau


def setups(max_days: float, quick: bool):
    days = [0.25, 0.5, 1, 2, 4, 8, 16, 32, 64, 128, 256, 365]
    if quick:
        days = [0.25, 0.5, 1, 4, 16, 64]
    out = []
    for d in days:
        if d > max_days:
            continue
        n_sft = int(round(d * 86400 / TSFT))
        if n_sft < 6:
            continue
        # the paper's timing runs: overlapping case
        out.append(("overlap", n_sft, _Grid(0, TSFT, n_sft - 2, 2 * TSFT, TSFT, n_sft - 1)))
        # embedded: t0 in the first half, tau up to a quarter of the data
        if n_sft >= 16:
            out.append(("embedded", n_sft, _Grid(0, TSFT, n_sft // 2, 2 * TSFT, TSFT,
                                                 max(n_sft // 4 - 1, 1))))
        # many t0, few tau, and the reverse: decouples N_sums from N_t0 N_tau
        if n_sft >= 64:
            out.append(("wide_t0", n_sft, _Grid(0, TSFT, n_sft // 2, 2 * TSFT, 8 * TSFT,
                                                max(n_sft // 32, 1))))
            out.append(("wide_tau", n_sft, _Grid(0, 16 * TSFT, max(n_sft // 32, 1), 2 * TSFT, TSFT,
                                                 n_sft // 4)))
    return out


def time_map(atoms, t, window, grid, min_ms: float = 20.0, reps: int = 5) -> float:
    """Median over `reps` CUDA-event intervals, each spanning enough back-to-back calls to exceed
    `min_ms` (SURVEY.md 8(d) timing protocol); seconds per call."""
    out_map = torch.empty((grid.N_t0, grid.N_tau), dtype=torch.float32, device="cuda")
    # the model is the paper's: the exponential window as the direct ("brute-force") sum, and ONE
    # code path per window (rect_method = 1: no one-launch small-map kernel, whose fixed cost is
    # half that of the three-launch chain and would be booked on c_SFTs)
    ws = torch.empty(B.workspace_bytes(window, int(t.shape[0]), 1, grid, exp_method=B.EXP_DIRECT,
                                       rect_method=1), dtype=torch.uint8, device="cuda")
    fn = lambda: B.tfstat_map(atoms, t, window, grid, out_map=out_map, workspace=ws,  # noqa: E731
                              exp_method=B.EXP_DIRECT, rect_method=1)
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    fn()
    e1.record()
    torch.cuda.synchronize()
    inner = max(1, min(200, int(min_ms / max(e0.elapsed_time(e1), 1e-3))))
    samples = []
    for _ in range(reps):
        e0.record()
        for _ in range(inner):
            fn()
        e1.record()
        torch.cuda.synchronize()
        samples.append(e0.elapsed_time(e1) / inner)
    return statistics.median(samples) * 1e-3


def measure(max_days: float, quick: bool, verbose: bool = True):
    rows = []
    for name, n_sft, grid in setups(max_days, quick):
        cells = grid.N_t0 * grid.N_tau
        if cells * 4 > 6 << 30:
            continue
        atoms, t = _atoms(n_sft)
        for window, wname in ((B.RECT, "rect"), (B.EXP, "exp")):
            n_sums = B.count_terms(t, window, grid)
            if window == B.EXP and n_sums > 4e12:
                continue  # > ~1 s per call: skip
            sec = time_map(atoms, t, window, grid)
            rows.append(dict(setup=name, window=wname, n_sft=n_sft, N_t0=grid.N_t0,
                             N_tau=grid.N_tau, cells=cells, n_sums=n_sums, seconds=sec))
            if verbose:
                print(f"{name:9s} {wname:4s} N_SFT {n_sft:6d} cells {cells:11d} "
                      f"N_sums {n_sums:.3e}  {sec * 1e6:10.1f} us", file=sys.stderr)
    return rows


def fit(rows):
    """The paper's three-step fit with the extra constant c_call."""
    R = [r for r in rows if r["window"] == "rect"]
    E = [r for r in rows if r["window"] == "exp"]
    short = [r for r in rows if r["cells"] <= 4096]
    c_sums_r = c_F = c_sums_e = 0.0
    # "in the following iterative steps to ensure convergence": the steps are
    # repeated with the later terms subtracted from the short-data-set times of step (i)
    for _ in range(6):
        # (i) short data sets: c_call + c_SFTs N_SFT
        A = np.array([[1.0, r["n_sft"]] for r in short])
        y = np.array([r["seconds"] - c_F * r["cells"] -
                      (c_sums_r if r["window"] == "rect" else c_sums_e) * r["n_sums"]
                      for r in short])
        (c_call, c_sfts), *_ = np.linalg.lstsq(A, y, rcond=None)
        c_sfts = max(c_sfts, 0.0)
        # (ii) rect: c_sums^r N_sums^r + c_F N_t0 N_tau; relative residuals (times span decades)
        yr = np.array([r["seconds"] - c_call - c_sfts * r["n_sft"] for r in R])
        Ar = np.array([[r["n_sums"], r["cells"]] for r in R], dtype=np.float64)
        w = 1.0 / np.array([r["seconds"] for r in R])
        (c_sums_r, c_F), *_ = np.linalg.lstsq(Ar * w[:, None], yr * w, rcond=None)
        c_sums_r, c_F = max(c_sums_r, 0.0), max(c_F, 0.0)
        # (iii) exp: c_sums^e N_sums^e
        ye = np.array([r["seconds"] - c_call - c_sfts * r["n_sft"] - c_F * r["cells"] for r in E])
        xe = np.array([r["n_sums"] for r in E], dtype=np.float64)
        we = 1.0 / np.array([r["seconds"] for r in E])
        c_sums_e = float(np.sum(we * we * xe * ye) / np.sum(we * we * xe * xe))

    def model(r):
        c = c_sums_r if r["window"] == "rect" else c_sums_e
        return c_call + c_sfts * r["n_sft"] + c * r["n_sums"] + c_F * r["cells"]

    rel = {wn: float(np.median([abs(model(r) - r["seconds"]) / r["seconds"]
                                for r in rows if r["window"] == wn])) for wn in ("rect", "exp")}
    # the asymptotic constants from the largest runs alone (where the fixed costs vanish)
    big_e = max(E, key=lambda r: r["n_sums"])
    big_r = max(R, key=lambda r: r["cells"])
    return dict(c_call=float(c_call), c_SFTs=float(c_sfts), c_sums_r=float(c_sums_r),
                c_F=float(c_F), c_sums_e=c_sums_e,
                c_r_PGM=float(c_sums_r + c_F), c_e_PGM=float(3.0 * c_sums_e),
                median_relative_residual=rel,
                largest_exp_run=dict(n_sums=big_e["n_sums"], seconds=big_e["seconds"],
                                     seconds_per_term=big_e["seconds"] / big_e["n_sums"]),
                largest_rect_run=dict(cells=big_r["cells"], seconds=big_r["seconds"],
                                      seconds_per_cell=big_r["seconds"] / big_r["cells"]),
                paper_table1={"Xeon E5-2630 LALPulsar": dict(c_r=3.4e-8, c_e=5.7e-8),
                              "GTX-1080(Ti) pyCUDA": dict(c_r=4.4e-9, c_e=6.2e-10),
                              "Tesla V100 pyCUDA": dict(c_r=4.3e-9, c_e=4.6e-11)})


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--out", default=None, help="write the measurements and the fit as JSON")
    ap.add_argument("--max-days", type=float, default=365.0)
    ap.add_argument("--quick", action="store_true")
    args = ap.parse_args(argv)
    B.load_library()
    rows = measure(args.max_days, args.quick)
    res = dict(gpu=torch.cuda.get_device_name(0), T_SFT=TSFT, fit=fit(rows), runs=rows)
    print(json.dumps(res["fit"], indent=1))
    if args.out:
        with open(args.out, "w") as f:
            json.dump(res, f, indent=1)
    return 0


if __name__ == "__main__":
    sys.exit(main())
