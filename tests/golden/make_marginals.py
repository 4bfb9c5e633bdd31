"""Writes the oracle's marginals of the FULL maps of BASELINE.json configs 4 and 5.

    python -m tests.golden.make_marginals [cfg5_rect] [cfg5_exp] [cfg4_exp]     (no argument: all)

Calls only `oracle/` (the fp64 CPU definitions) and `synth/` (the seeded input generators); no
value comes from the CUDA path.  The full maps are too slow for the test suite (config 5:
5.4e10 / 7.2e10 window-atom terms per window; config 4: 1.08e12 over 4096 templates, about half
an hour on 8 cores), so their marginals are computed once here and stored as text next to this
script; tests/test_gpu_parity.py compares the GPU's fused marginals with them (SURVEY.md 8(c)/(d):
"check parity on all 4096 once (cache oracle results on disk keyed by seed)").

File format (load_golden.load): one `key v1 v2 ...` line per quantity.
  seed        the synth seed of the workload (synth.atoms.BASE_SEED + config id)
  max2F m n logB n_valid          one value per template, in template order
  runner_up   per template: the largest 2F of the map that is NOT at (m, n) (config 5 only; lets
              the test accept another argmax only on a tie within the 2F tolerance)
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from synth import make_workload  # noqa: E402
from synth.atoms import BASE_SEED  # noqa: E402

RECT, EXP = 0, 1


def _write(name, config_id, rows, runner_up=None):
    path = os.path.join(HERE, name)
    with open(path, "w") as f:
        f.write(f"# written by tests/golden/make_marginals.py from oracle/ (fp64) on synth config {config_id}\n")
        f.write(f"seed {BASE_SEED + config_id}\n")
        f.write("max2F " + " ".join(f"{r.max2F:.17g}" for r in rows) + "\n")
        f.write("m " + " ".join(str(r.m) for r in rows) + "\n")
        f.write("n " + " ".join(str(r.n) for r in rows) + "\n")
        f.write("logB " + " ".join(f"{r.logB:.17g}" for r in rows) + "\n")
        f.write("n_valid " + " ".join(str(r.n_valid) for r in rows) + "\n")
        if runner_up is not None:
            f.write("runner_up " + " ".join(f"{v:.17g}" for v in runner_up) + "\n")
    print("wrote", path, flush=True)


def cfg5(window, name):
    wl = make_workload(5)
    t0 = time.time()
    ref = oracle.map2F(wl.data.atoms[0], wl.data.t, window, wl.grid)
    mg = oracle.marginalise(ref["twoF"], ref["flags"])
    v = np.where(ref["flags"] == 0, ref["twoF"], -np.inf)
    v[mg.m, mg.n] = -np.inf
    print(f"{name}: oracle full map in {time.time() - t0:.0f} s, {int(ref['cnt'].sum())} terms",
          flush=True)
    _write(name, 5, [mg], [float(v.max())])


def cfg4(name):
    wl = make_workload(4)
    rows = []
    t0 = time.time()
    step = 64
    for k0 in range(0, wl.n_templates, step):
        res, _ = oracle.search(wl.data.atoms[k0:k0 + step], wl.data.t, EXP, wl.grid)
        rows.extend(res)
        print(f"{name}: {k0 + step}/{wl.n_templates} templates, {time.time() - t0:.0f} s",
              flush=True)
    _write(name, 4, rows)


if __name__ == "__main__":
    todo = sys.argv[1:] or ["cfg5_rect", "cfg5_exp", "cfg4_exp"]
    if "cfg5_rect" in todo:
        cfg5(RECT, "cfg5_rect_marginals.txt")
    if "cfg5_exp" in todo:
        cfg5(EXP, "cfg5_exp_marginals.txt")
    if "cfg4_exp" in todo:
        cfg4("cfg4_exp_marginals.txt")
