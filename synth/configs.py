"""The five BASELINE.json workloads as seeded synthetic inputs, plus tiny cases.

config ids are 1-based like SURVEY.md section 8(d): config k == BASELINE.json
configs[k-1].  t0_min = 0 = data start in every config.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

from .atoms import (TSFT, AtomSet, Grid, gap_mask, inject_exponential,
                    make_atoms, pack_atoms, template_seed)

DAY = 86400
RECT, EXP = 0, 1

CONFIGS: Dict[int, dict] = {
    1: dict(name="cfg1_rect_48atoms_24x24", windows=(RECT,), n_slots=48, gaps=0.0,
            grid=Grid(0, TSFT, 24, TSFT, TSFT, 24), n_templates=1),
    2: dict(name="cfg2_exp_1440atoms_480x937_inj", windows=(EXP,), n_slots=1440,
            gaps=0.0, grid=Grid(0, TSFT, 480, DAY // 2, TSFT, 937), n_templates=1,
            inject=dict(t0=4 * DAY, tau=6 * DAY, rho=10.0)),
    3: dict(name="cfg3_glitch_4608atoms_96x5736", windows=(EXP, RECT), n_slots=5760,
            gaps=0.20, grid=Grid(0, TSFT, 96, DAY // 2, TSFT, 5736), n_templates=1),
    4: dict(name="cfg4_search_4096x2880atoms_96x1417", windows=(EXP,), n_slots=2880,
            gaps=0.0, grid=Grid(0, TSFT, 96, DAY // 2, TSFT, 1417), n_templates=4096,
            inject_frac=0.01, inject_rho=8.0),
    5: dict(name="cfg5_year_13140atoms_17520x720", windows=(RECT, EXP),
            n_slots=17520, gaps=0.25, grid=Grid(0, TSFT, 17520, DAY // 2, DAY // 2, 720),
            n_templates=1),
}


@dataclass
class Workload:
    config_id: int
    name: str
    windows: Tuple[int, ...]
    grid: Grid
    data: AtomSet
    templates: np.ndarray  # global template indices held in `data`
    # injected cells: template index -> (m, n, rho)
    injections: Dict[int, Tuple[int, int, float]] = field(default_factory=dict)

    @property
    def n_templates(self) -> int:
        return self.data.n_templates


def _timestamps(cfg: dict, config_id: int) -> np.ndarray:
    n_slots = cfg["n_slots"]
    slots = np.arange(n_slots, dtype=np.int64)
    if cfg["gaps"] > 0.0:
        rng = np.random.default_rng(template_seed(config_id, 1 << 30))
        slots = slots[gap_mask(n_slots, cfg["gaps"], rng)]
    return (slots * TSFT).astype(np.int32)


def cfg4_injection_plan(config_id: int = 4) -> Dict[int, Tuple[int, int, float]]:
    """Which of the 4096 templates carry a signal, and at which grid cell."""
    cfg = CONFIGS[config_id]
    g: Grid = cfg["grid"]
    rng = np.random.default_rng(template_seed(config_id, (1 << 30) + 1))
    n_inj = int(round(cfg["inject_frac"] * cfg["n_templates"]))
    idx = np.sort(rng.choice(cfg["n_templates"], size=n_inj, replace=False))
    ms = rng.integers(0, g.N_t0, size=n_inj)
    ns = rng.integers(0, g.N_tau, size=n_inj)
    return {int(i): (int(m), int(n), float(cfg["inject_rho"]))
            for i, m, n in zip(idx, ms, ns)}


def make_workload(config_id: int,
                  templates: Optional[Sequence[int]] = None) -> Workload:
    """Build config `config_id`.  `templates` selects a subset of global template
    indices (config 4 only; each template has its own seed, so a subset is
    bit-identical to the same templates inside the full set)."""
    cfg = CONFIGS[config_id]
    g: Grid = cfg["grid"]
    t = _timestamps(cfg, config_id)
    if templates is None:
        templates = range(cfg["n_templates"])
    templates = np.asarray(list(templates), dtype=np.int64)
    plan: Dict[int, Tuple[int, int, float]] = {}
    if "inject_frac" in cfg:
        plan = cfg4_injection_plan(config_id)
    per_template: List[np.ndarray] = []
    injections: Dict[int, Tuple[int, int, float]] = {}
    for k in templates:
        rng = np.random.default_rng(template_seed(config_id, int(k)))
        phi = float(rng.uniform(0.0, 2.0 * np.pi)) if config_id == 4 else 0.0
        a32 = make_atoms(t, rng, phi=phi).astype(np.float32)
        if "inject" in cfg:
            inj = cfg["inject"]
            inject_exponential(a32, t, inj["t0"], inj["tau"], inj["rho"], rng)
            m = (inj["t0"] - g.t0_min) // g.dt0
            n = (inj["tau"] - g.tau_min) // g.dtau
            injections[int(k)] = (int(m), int(n), float(inj["rho"]))
        if int(k) in plan:
            m, n, rho = plan[int(k)]
            inject_exponential(a32, t, g.t0_min + m * g.dt0, g.tau_min + n * g.dtau,
                               rho, rng)
            injections[int(k)] = (m, n, rho)
        per_template.append(a32)
    return Workload(config_id, cfg["name"], tuple(cfg["windows"]), g,
                    AtomSet(pack_atoms(per_template), t), templates, injections)


def tiny_workload(seed: int, n_slots: int, gaps: float, grid: Grid,
                  n_templates: int = 1, phi_random: bool = False) -> Workload:
    """Small seeded case with the same atom model, for tests that span several
    tiles and a ragged tail but finish in seconds in the oracle."""
    ss = np.random.SeedSequence(seed)
    slots = np.arange(n_slots, dtype=np.int64)
    if gaps > 0.0:
        slots = slots[gap_mask(n_slots, gaps, np.random.default_rng(ss.spawn(1)[0]),
                               mean_len=4.0)]
    t = (slots * TSFT).astype(np.int32)
    per_template = []
    for child in ss.spawn(n_templates):
        rng = np.random.default_rng(child)
        phi = float(rng.uniform(0.0, 2.0 * np.pi)) if phi_random else 0.0
        per_template.append(make_atoms(t, rng, phi=phi).astype(np.float32))
    return Workload(0, f"tiny_seed{seed}", (RECT, EXP), grid,
                    AtomSet(pack_atoms(per_template), t),
                    np.arange(n_templates, dtype=np.int64))
