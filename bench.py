#!/usr/bin/env python
"""bench.py -- throughput of the transient F-statistic hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path (bounds, exp-window
weighted sums, cell closure, fused marginalisation, batched over templates) over one batch of
synthetic input: BASELINE.json configs[3], the batched template search (4096 templates x 2880
atoms, 96 x 1417 grid, 1.078e12 window-atom terms), through tfstat_search of the C ABI.
Prints ONE JSON line (see DESIGN.md "Measurement" for every field).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "exp-window window-atom terms/s"
UNIT = "terms/s"
WORKLOAD = "cfg4_search_4096x2880atoms_96x1417"
# algorithmic work per window-atom term: 1 FFMA (exp argument) + 1 FMUL (w^2)
# + 7 FFMA (A,B,C,Re/Im Fa,Re/Im Fb) on the FP32 pipe, + 1 MUFU.EX2 on the XU pipe
FP32_OPS_PER_TERM = 9
FP32_LANES_PER_CLK_SM = 128  # cc 10.0: 4 SMSPs x 32 FP32 lanes
# dram__bytes_read.sum + dram__bytes_write.sum of exp_direct_kernel, 296 templates of config 4
NCU_CAPTURE = "profiles/r02_exp_direct_full.md"
NCU_DRAM_BYTES_PER_TEMPLATE = (51.410176e6 + 1.434368e6) / 296
PACK_BLOCK = 768  # kPackBlock of csrc/tfstat_dev.cuh: packed records are padded to whole blocks


def plan_packed_bytes(n_atoms: int, n_templates: int) -> int:
    """Bytes of packed atom records (32 B per atom) the exponential-window kernels stream."""
    n_pad = (n_atoms + PACK_BLOCK - 1) // PACK_BLOCK * PACK_BLOCK
    return 32 * n_pad * n_templates


def read_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md)."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows = []
        self.proc = None
        self.gpu_index = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-i", str(self.gpu_index), "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, power, reasons = [], [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[1]))
                smax.append(float(r[2]))
                power.append(float(r[3]))
            except (ValueError, IndexError):
                continue
            for name, col in (("hw_slowdown", 5), ("hw_thermal_slowdown", 6),
                              ("sw_thermal_slowdown", 7), ("sw_power_cap", 8)):
                if len(r) > col and r[col].lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # "under load": samples in the upper half of the power range seen
        thr = 0.5 * (max(power) + min(power))
        load = [s for s, p in zip(sm, power) if p >= thr] or sm
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": max(smax),
                "power_w_max": max(power), "samples": len(sm), "reasons": sorted(reasons)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    return rank, local, world


# ------------------------------------------------------------------------------------------
# reference arm: the fp64 oracle as it stands, on the host cores
# ------------------------------------------------------------------------------------------
def oracle_leg(n_templates: int, seed_offset: int = 0, n_threads: int = 0):
    """Times oracle.search on `n_templates` templates of config 4.  Returns
    (terms_per_s, seconds, terms, cores)."""
    import oracle
    from synth import make_workload

    wl = make_workload(4, templates=range(seed_offset, seed_offset + n_templates))
    cores = n_threads if n_threads > 0 else oracle.num_threads()
    t0 = time.perf_counter()
    _, terms = oracle.search(wl.data.atoms, wl.data.t, 1, wl.grid, n_threads=cores)
    dt = time.perf_counter() - t0
    return terms / dt, dt, terms, min(cores, n_templates)


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    import oracle

    cores = oracle.num_threads()
    n_tpl = max(1, min(cores, 16))  # one template (2.6e8 terms, a few seconds) per core
    n_warm = min(args.warmup, 1)  # one 1-template pass (pages in the library and the inputs);
    for _ in range(n_warm):        # more would only burn host-core minutes: nothing here is cached
        oracle_leg(1)
    times, terms = [], 0
    for s in range(args.steps):
        _, dt, terms, used = oracle_leg(n_tpl, seed_offset=s * n_tpl)
        times.append(dt)
    ms = 1e3 * sum(times) / len(times)
    value = terms / (ms * 1e-3)
    sample = (f"{n_tpl} of 4096 templates of config 4 per step (full 96x1417 grid each, "
              f"{terms:.3e} terms), OpenMP over templates")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": n_warm, "warmup_requested": args.warmup,
        "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": min(cores, n_tpl),
                         "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------
def time_calls(torch, fn, n, stream=None):
    """CUDA-event time of n back-to-back calls on the current stream, ms per call."""
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(n):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n


def side_workloads(torch, pkg, peaks):
    """Kernel-level numbers for the other BASELINE.json configs (context, not the bench line)."""
    from synth import make_workload

    out = {}
    l2_flush = torch.empty(192 << 20, dtype=torch.uint8, device="cuda")

    def timed(fn, reps=5):
        ms = []
        for _ in range(reps):
            l2_flush.zero_()
            ms.append(time_calls(torch, fn, 1))
        return min(ms), statistics.median(ms)

    for cfg, window, wname in ((2, 1, "exp"), (3, 1, "exp"), (3, 0, "rect"), (5, 0, "rect"),
                               (5, 1, "exp")):
        wl = make_workload(cfg)
        atoms = torch.from_numpy(wl.data.atoms).cuda()
        t = torch.from_numpy(wl.data.t).cuda()
        terms = pkg.count_terms(t, window, wl.grid)
        cells = wl.grid.n_cells
        ws = torch.empty(pkg.workspace_bytes(window, t.shape[0], 1, wl.grid,
                                             exp_method=pkg.EXP_DIRECT), dtype=torch.uint8,
                         device="cuda")
        maps = torch.empty((wl.grid.N_t0, wl.grid.N_tau), dtype=torch.float32, device="cuda")
        fn_map = lambda: pkg.tfstat_map(atoms[0], t, window, wl.grid, out_map=maps, workspace=ws,
                                        exp_method=pkg.EXP_DIRECT)
        fn_fused = lambda: pkg.tfstat_search(atoms, t, window, wl.grid, workspace=ws,
                                             exp_method=pkg.EXP_DIRECT)
        for _ in range(3):
            fn_map()
            fn_fused()
        best_map, med_map = timed(fn_map)
        best_fused, med_fused = timed(fn_fused)
        rec = {"cells": cells, "terms": terms, "map_ms": med_map, "fused_marginals_ms": med_fused}
        if window == 1:
            rec["terms_per_s_map"] = terms / (med_map * 1e-3)
            rec["terms_per_s_fused"] = terms / (med_fused * 1e-3)
            # the same map through the DEFAULT form (EXP_AUTO = the exact sliding form, DESIGN.md
            # 6.2): what a caller gets without options; EFFECTIVE terms/s (A.6 count / time)
            ws_a = torch.empty(pkg.workspace_bytes(window, t.shape[0], 1, wl.grid),
                               dtype=torch.uint8, device="cuda")
            fn_auto = lambda: pkg.tfstat_map(atoms[0], t, window, wl.grid, out_map=maps,
                                             workspace=ws_a)
            for _ in range(3):
                fn_auto()
            _, med_auto = timed(fn_auto)
            rec["default_form_map_ms"] = med_auto
            rec["default_form_effective_terms_per_s"] = terms / (med_auto * 1e-3)
            rec["default_form_plan"] = pkg.plan_info(window, int(t.shape[0]), 1, wl.grid)
        else:
            by = 32 * int(t.shape[0]) + 4 * cells  # atoms once + 4 B per cell
            rec["cells_per_s_map"] = cells / (med_map * 1e-3)
            rec["algorithmic_GBps_map"] = by / (med_map * 1e-3) / 1e9
            rec["hbm_frac_map"] = rec["algorithmic_GBps_map"] / peaks["hbm_gbs"]
            # the same call captured ONCE in a CUDA graph and replayed (what a caller in a loop
            # does with a launch-bound call: a cold single call above pays the host's launch
            # latency of every kernel of the chain, the replay only the chain itself)
            a1 = atoms[0]
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                fn_map()
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                pkg.tfstat_map(a1, t, window, wl.grid, out_map=maps, workspace=ws)
            _, med_graph = timed(graph.replay)
            rec["map_graph_replay_ms"] = med_graph
            rec["hbm_frac_map_graph_replay"] = by / (med_graph * 1e-3) / 1e9 / peaks["hbm_gbs"]
            del graph
        if cfg == 2:
            # the same map through tfstat_map_general (explicit grid arrays, one weight per term:
            # the paper's own brute-force design), exp and a 1025-point table
            t0g = torch.from_numpy(wl.grid.t0().astype(np.int32)).cuda()
            taug = torch.from_numpy(wl.grid.tau().astype(np.int32)).cuda()
            tab = torch.exp(-torch.linspace(0.0, 3.0, 1025, device="cuda"))
            for gname, kind, tb in (("exp", 1, None), ("table", 2, tab)):
                fn_g = lambda: pkg.tfstat_map_general(atoms[0], t, kind, (3, 1), t0g, taug,
                                                      table=tb, want_marginals=False)
                for _ in range(3):
                    fn_g()
                _, med_g = timed(fn_g)
                rec[f"general_{gname}_map_ms"] = med_g
                rec[f"general_{gname}_terms_per_s"] = terms / (med_g * 1e-3)
        out[f"cfg{cfg}_{wname}"] = rec
        if cfg == 5 and window == 0:
            # steady state of the rect map path: 8 copies of config 5 in one tfstat_search that
            # writes all maps (404 MB > L2), so launch latency and the single-wave tail of the
            # one-template call are amortised
            T8 = 8
            a8 = atoms.expand(T8, -1, -1).contiguous()
            ws8 = torch.empty(pkg.workspace_bytes(0, int(t.shape[0]), T8, wl.grid),
                              dtype=torch.uint8, device="cuda")
            res8 = [None]

            def fn8():
                res8[0] = pkg.tfstat_search(a8, t, 0, wl.grid, workspace=ws8, want_maps=True)

            fn8()
            maps8 = res8[0].maps

            def fn8b():  # reuse the output tensor: no allocation inside the timed call
                lib = pkg.load_library()
                o = res8[0].raw
                rc = lib.tfstat_search(a8.data_ptr(), a8.stride(0), a8.stride(1), t.data_ptr(),
                                       int(t.shape[0]), T8, 0, wl.grid.t0_min, wl.grid.dt0,
                                       wl.grid.N_t0, wl.grid.tau_min, wl.grid.dtau, wl.grid.N_tau,
                                       o.data_ptr(), maps8.data_ptr(), None, ws8.data_ptr(),
                                       ws8.numel(), torch.cuda.current_stream().cuda_stream, None)
                assert rc == 0

            fn8b()
            ms8 = time_calls(torch, fn8b, 5)
            by8 = T8 * by
            out["cfg5x8_rect_maps"] = {"templates": T8, "ms": ms8,
                                       "algorithmic_GBps": by8 / (ms8 * 1e-3) / 1e9,
                                       "hbm_frac": by8 / (ms8 * 1e-3) / 1e9 / peaks["hbm_gbs"]}
            del a8, ws8, maps8, res8
        # marginalise-from-HBM (row a5 standalone), HBM-bound: 4 B per cell read
        if cfg == 5 and window == 0:
            fn_m = lambda: pkg.tfstat_marginalise(maps)
            for _ in range(3):
                fn_m()
            b, med = timed(fn_m)
            out["cfg5_marginalise"] = {"cells": cells, "ms": med,
                                       "algorithmic_GBps": 4 * cells / (med * 1e-3) / 1e9,
                                       "hbm_frac": 4 * cells / (med * 1e-3) / 1e9 / peaks["hbm_gbs"]}
            # the same two kernels through the entry point that allocates nothing, captured in a
            # CUDA graph and replayed: the device chain without the host's share of a single call
            out_m = torch.empty((1, 5), dtype=torch.int32, device="cuda")
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                pkg.tfstat_marginalise_static(maps, out=out_m)
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            graph_m = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph_m):
                pkg.tfstat_marginalise_static(maps, out=out_m)
            _, med_g = timed(graph_m.replay)
            out["cfg5_marginalise"]["graph_replay_ms"] = med_g
            out["cfg5_marginalise"]["hbm_frac_graph_replay"] = (
                4 * cells / (med_g * 1e-3) / 1e9 / peaks["hbm_gbs"])
            del graph_m
    # config 1 (24 x 24 cells, 48 atoms; Fig. 3's one-day data set): one launch of
    # the small-map kernel; and the same shape x 1000 seeded templates (Fig. 3's 1000 bins)
    from synth import Grid as _G, tiny_workload as _tw
    wl1 = make_workload(1)
    a1 = torch.from_numpy(wl1.data.atoms).cuda()
    t1 = torch.from_numpy(wl1.data.t).cuda()
    ws1 = torch.empty(pkg.workspace_bytes(0, 48, 1000, wl1.grid), dtype=torch.uint8, device="cuda")
    fn1 = lambda: pkg.tfstat_search(a1, t1, 0, wl1.grid, workspace=ws1, want_maps=True)
    wlk = _tw(11, 48, 0.0, _G(0, 1800, 24, 1800, 1800, 24), n_templates=1000, phi_random=True)
    ak = torch.from_numpy(wlk.data.atoms).cuda()
    fnk = lambda: pkg.tfstat_search(ak, t1, 0, wl1.grid, workspace=ws1)
    for _ in range(3):
        fn1()
        fnk()
    out["cfg1_rect"] = {"cells": wl1.grid.n_cells, "map_and_marginals_ms": timed(fn1)[1],
                        "x1000_templates_fused_ms": time_calls(torch, fnk, 10),
                        "note": "one launch (rect_small_kernel); single-call time is host-launch bound"}
    out["cfg1_rect"]["x1000_cells_per_s"] = 576e3 / (out["cfg1_rect"]["x1000_templates_fused_ms"] * 1e-3)
    # per-detector merge at config-4 scale: 2 detectors x 1024 templates x 2880 atoms, each with
    # ~20 % of its own slots missing, merged onto the union (HBM-bound: reads both sets once,
    # writes the merged set once)
    n_at, T_m = 2880, 1024
    tt = torch.arange(n_at, device="cuda", dtype=torch.int32) * 1800
    gen = torch.Generator(device="cuda").manual_seed(5)
    keep = [torch.rand(n_at, generator=gen, device="cuda") > 0.2 for _ in range(2)]
    t_d = [tt[k].contiguous() for k in keep]
    a_d = [torch.randn((T_m, 7, int(x.shape[0])), generator=gen, device="cuda") for x in t_d]
    t_u = torch.unique(torch.cat(t_d)).to(torch.int32).contiguous()
    fn_mg = lambda: pkg.tfstat_merge_detectors(a_d, t_d, t_u)
    for _ in range(3):
        fn_mg()
    ms_mg = time_calls(torch, fn_mg, 10)
    by_mg = 4 * (sum(a.numel() for a in a_d) + T_m * 7 * int(t_u.shape[0]))
    out["merge_detectors_2x1024x2880"] = {"ms": ms_mg, "algorithmic_GBps": by_mg / (ms_mg * 1e-3) / 1e9,
                                          "hbm_frac": by_mg / (ms_mg * 1e-3) / 1e9 / peaks["hbm_gbs"]}
    del a_d
    # row a5 standalone at a size where the two-launch chain is amortised: the map of one year at
    # dt0 = dtau = T_SFT (17518 x 17519 cells, 1.23 GB), the largest of the paper's setups
    # (PAPER.md:106, 146-148); values are arbitrary positive floats, the kernel is data-independent
    big = torch.rand((17518, 17519), device="cuda") * 8.0
    fn_b = lambda: pkg.tfstat_marginalise(big)
    for _ in range(3):
        fn_b()
    ms_b = time_calls(torch, fn_b, 10)
    out["marginalise_1yr_full_resolution"] = {
        "cells": big.numel(), "ms": ms_b, "algorithmic_GBps": 4 * big.numel() / (ms_b * 1e-3) / 1e9,
        "hbm_frac": 4 * big.numel() / (ms_b * 1e-3) / 1e9 / peaks["hbm_gbs"],
        "l2": "1.23 GB per call > 126 MB L2, no flush"}
    # rows a2-a4 at the same size: the rectangular map of one year of gapless SFTs at dt0 = dtau =
    # T_SFT, written into the same 1.23 GB buffer; once with N_tau = 17519 (rows not 16-byte
    # aligned: scalar coalesced write-out) and once with N_tau = 17516 (vector write-out)
    from synth.atoms import Grid as SGrid, make_atoms
    n_y = 17520
    t_y = np.arange(n_y, dtype=np.int64) * 1800
    at_y = torch.from_numpy(make_atoms(t_y, np.random.default_rng(11)).astype(np.float32)).cuda()
    tt_y = torch.from_numpy(t_y.astype(np.int32)).cuda()
    leg = {}
    for n_tau in (n_y - 1, n_y - 4):
        g_y = SGrid(0, 1800, n_y - 2, 3600, 1800, n_tau)
        m_y = big.view(-1)[: g_y.n_cells].view(g_y.N_t0, g_y.N_tau)
        ws_y = torch.empty(pkg.workspace_bytes(pkg.RECT, n_y, 1, g_y, rect_method=1),
                           dtype=torch.uint8, device="cuda")
        fn_y = lambda: pkg.tfstat_map(at_y, tt_y, pkg.RECT, g_y, out_map=m_y, workspace=ws_y,
                                      rect_method=1)
        for _ in range(3):
            fn_y()
        ms_y = time_calls(torch, fn_y, 10)
        leg[f"N_tau_{n_tau}"] = {"cells": g_y.n_cells, "ms": ms_y,
                                 "algorithmic_GBps": 4 * g_y.n_cells / (ms_y * 1e-3) / 1e9,
                                 "hbm_frac": 4 * g_y.n_cells / (ms_y * 1e-3) / 1e9 / peaks["hbm_gbs"]}
    out["rect_map_1yr_full_resolution"] = leg
    del big
    return out


def run_ours(args):
    import torch

    import paper_1805_05652_b200 as pkg
    from synth import make_workload

    rank, local, world = dist_env()
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("--gpus N > 1 must be launched with torch.distributed.run")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    pkg.load_library()  # no fallback: raises if libtfstat.so is missing
    peaks = read_peaks()

    n_tpl = args.templates
    # weak scaling: every rank searches its own n_tpl templates (distinct seeds), no data-path
    # collective
    wl = make_workload(4, templates=range(rank * n_tpl, rank * n_tpl + n_tpl))
    grid = wl.grid
    atoms_h = torch.from_numpy(wl.data.atoms).pin_memory()
    t_h = torch.from_numpy(wl.data.t).pin_memory()
    atoms = atoms_h.cuda()
    t = t_h.cuda()
    terms_per_template = pkg.count_terms(t, pkg.EXP, grid)
    terms = terms_per_template * n_tpl
    cells = grid.n_cells * n_tpl
    ws = torch.empty(pkg.workspace_bytes(pkg.EXP, int(t.shape[0]), n_tpl, grid,
                                         exp_method=pkg.EXP_DIRECT),
                     dtype=torch.uint8, device="cuda")
    out = torch.empty((n_tpl, 5), dtype=torch.int32, device="cuda")

    def step(events=None):
        # the headline is the DIRECT truncated sum (real window-atom terms); the library's
        # default (EXP_AUTO) is the sliding form, reported as other_workloads.cfg4_exp_scan
        return pkg.tfstat_search(atoms, t, pkg.EXP, grid, workspace=ws, out=out,
                                 main_kernel_events=events, exp_method=pkg.EXP_DIRECT)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()

    # ---- device-resident timing: exactly K steps, barrier + sync on both sides ----------
    kernel_events = []
    for _ in range(args.steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        b.record()
        kernel_events.append((a, b))
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(args.steps):
        step(kernel_events[k])
    e1.record()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_total = e0.elapsed_time(e1)
    kernel_ms = [a.elapsed_time(b) for a, b in kernel_events]
    if dist:
        tt = torch.tensor([ms_total], device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms_total = float(tt.item())
    ms_per_step = ms_total / args.steps
    value = terms * world / (ms_per_step * 1e-3)
    res_dev = out.cpu().numpy().copy()

    # ---- end to end through the C ABI with HOST buffers (H2D + compute + D2H inside) -----
    for _ in range(max(args.warmup, 3)):
        pkg.tfstat_search_host(atoms_h, t_h, pkg.EXP, grid, exp_method=pkg.EXP_DIRECT)
    if dist:
        dist.barrier()
    t0 = time.perf_counter()
    e2e_each = []
    for _ in range(args.steps):
        t1 = time.perf_counter()
        res_host, _ = pkg.tfstat_search_host(atoms_h, t_h, pkg.EXP, grid, exp_method=pkg.EXP_DIRECT)
        e2e_each.append((time.perf_counter() - t1) * 1e3)
    e2e_s = (time.perf_counter() - t0) / args.steps
    if os.environ.get("TFSTAT_BENCH_VERBOSE"):
        print("e2e ms per call:", [round(x, 1) for x in e2e_each], file=sys.stderr)
    if dist:
        tt = torch.tensor([e2e_s], device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e_s = float(tt.item())
    assert np.array_equal(res_host.view(np.int32).reshape(-1, 5), res_dev), \
        "host-buffer path and device-resident path disagree"
    h2d = atoms_h.numel() * 4 + t_h.numel() * 4
    d2h = n_tpl * 20

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (exp_direct_kernel) -----------------------------
    k_ms = statistics.mean(kernel_ms)
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    peak_ops = FP32_LANES_PER_CLK_SM * n_sm * peaks["sm_max_mhz"] * 1e6  # lane-ops/s at max clock
    # The kernel shares one weight among the C cells of a t0 tile (eq. 7 is invariant to the
    # per-cell factor) and takes its square from a second MUFU.EX2 (ALU + XU pipes) instead of a
    # multiply, so it EXECUTES 7 + 1/C FP32 lane-ops per term (the 7 multiply-adds and the weight's
    # argument), not the algorithmic 9.
    # "the roofline fraction is always computed from the executed mix, while
    # terms/s always uses the A.6 count" -- so `achieved` / `frac` are the executed ones (<= 1 by
    # construction) and the 9-op algorithmic figures are given beside them (they can exceed 1).
    # C is what the library ran (tfstat_plan_info), not a copy of its rule.
    plan = pkg.plan_info(pkg.EXP, int(t.shape[0]), n_tpl, grid, exp_method=pkg.EXP_DIRECT)
    assert plan["kernel_name"] == "exp_direct"
    tile_c = plan["tile_c"]
    exec_ops_per_term = 7.0 + 1.0 / tile_c
    ach_ops = terms * exec_ops_per_term / (k_ms * 1e-3)
    alg_ops = terms * FP32_OPS_PER_TERM / (k_ms * 1e-3)
    probes = {k: pkg.probe_alu(k) for k in ("ffma", "fadd", "mufu_ex2", "ffma2", "ffma_mufu",
                                             "lds128", "dfma", "ffma2_two_pairs",
                                             "ffma2_scalar_pair", "ffma2_two_scalars")}
    roofline = {
        "bound": "alu", "kernel": "exp_direct_kernel",
        "achieved": ach_ops / 1e12, "peak": peak_ops / 1e12, "unit": "T FP32 lane-op/s",
        "frac": ach_ops / peak_ops,
        "peak_source": (f"{FP32_LANES_PER_CLK_SM} FP32 lanes/clk/SM x {n_sm} SMs x "
                        f"{peaks['sm_max_mhz']:.0f} MHz (max SM clock, {peaks['source']})"),
        "executed_ops_per_term": exec_ops_per_term, "tile_c": tile_c,
        "algorithmic_ops_per_term": FP32_OPS_PER_TERM,
        "achieved_algorithmic": alg_ops / 1e12, "frac_algorithmic": alg_ops / peak_ops,
        "note": ("achieved/frac count the EXECUTED FP32 lane-ops (7 + 1/C per term: one weight per "
                 "t0 tile of C cells, its square by a second MUFU.EX2 off the FP32 pipe -- which "
                 "made the kernel 1.3 % faster and this fraction 1.7 % smaller); *_algorithmic "
                 "charge 9 per term and can exceed 1"),
        "kernel_ms": k_ms, "kernel_share_of_step": k_ms / ms_per_step,
        "terms_per_s_kernel": terms / (k_ms * 1e-3),
        "terms_per_clk_sm": terms / (k_ms * 1e-3) / n_sm /
        ((clocks or {}).get("sm_mhz") or peaks["sm_max_mhz"]) / 1e6,
        "measured_ffma_lane_ops_per_s": probes["ffma"]["lane_ops_per_s"],
        "frac_of_measured_ffma": ach_ops / probes["ffma"]["lane_ops_per_s"],
        # NOT measured in this run: dram__bytes_read.sum + dram__bytes_write.sum of the kernel in
        # the ncu --set full capture NCU_CAPTURE (296 templates), scaled per template to this launch
        "traffic": NCU_DRAM_BYTES_PER_TEMPLATE * n_tpl,
        "traffic_unit": f"bytes per launch, scaled per template from the capture {NCU_CAPTURE}",
        "algorithmic_bytes": int(plan_packed_bytes(int(t.shape[0]), n_tpl)),
        "algorithmic_bytes_note": "the kernel reads the PACKED records (32 B per atom, padded to "
                                  "768 atoms); pack_atoms_kernel reads the caller's 28 B + writes them",
        "plan": plan,
        "probes_ops_per_clk_sm": {k: round(v["ops_per_clk_sm"], 2) for k, v in probes.items()},
        # the kernel's core loop with nothing around it, in the shipped accumulator layout (pairs
        # of cells: two broadcast-scalar multiplicands) and in round 1's (pairs of channels); and
        # with 2 / 4 more LDS.128 per atom whose results nobody uses (what do register
        # write-backs that are not accumulator updates cost the FMA stream? DESIGN.md 6.1)
        "isolated_core_loop_terms_per_clk_sm": {
            f"{d['form']}_c{d['cells']}": round(d["terms_per_clk_sm"], 2)
            for d in (pkg.probe_direct_loop(f, c) for f in (0, 1, 2, 3) for c in (8, 16))},
        "probe_sm_mhz": round(probes["ffma"]["sm_mhz"], 1),
    }

    # ---- CPU baseline: the oracle as it stands on this box's host cores -------------------
    cpu = None
    if not args.no_cpu_baseline:
        import oracle

        cores = oracle.num_threads()
        n_s = 5 * max(1, min(cores, 16))  # ~10 s of CPU work: 5 templates of 2.6e8 terms per core
        v, dt, tms, used = oracle_leg(n_s)
        v1, dt1, tms1, _ = oracle_leg(1, n_threads=1)  # comparable to Table 1's per-core constants
        cpu = {"value": v, "unit": UNIT, "cores": used, "kind": "oracle", "seconds": dt,
               "sample": f"{n_s} of 4096 templates of config 4 (full 96x1417 grid each, "
                         f"{tms:.3e} terms), OpenMP over templates",
               "single_core": {"value": v1, "unit": UNIT, "seconds": dt1,
                               "seconds_per_term": dt1 / tms1,
                               "sample": f"1 template, {tms1:.3e} terms, 1 thread"}}

    side = None if args.no_side else side_workloads(torch, pkg, peaks)
    if side is not None:
        # the same config-4 search through the exact factorised sliding form (TFSTAT_EXP_SCAN):
        # EFFECTIVE terms/s (the A.6 term count divided by the time; the kernel does ~60x fewer
        # weighted terms), checked against the direct results of the timed run
        ws_s = torch.empty(pkg.workspace_bytes(pkg.EXP, int(t.shape[0]), n_tpl, grid,
                                               exp_method=pkg.EXP_SCAN),
                           dtype=torch.uint8, device="cuda")
        out_s = torch.empty_like(out)
        fn_s = lambda: pkg.tfstat_search(atoms, t, pkg.EXP, grid, workspace=ws_s, out=out_s,
                                         exp_method=pkg.EXP_SCAN)
        for _ in range(2):
            fn_s()
        ms_s = time_calls(torch, fn_s, 3)
        r_s = out_s.cpu().numpy().view(pkg.RESULT_DTYPE).reshape(-1)
        r_d = res_dev.view(pkg.RESULT_DTYPE).reshape(-1)
        dmax = float(np.max(np.abs(r_s["max2F"] - r_d["max2F"]) / np.maximum(1.0, r_d["max2F"])))
        # and end to end from pinned host memory (what a caller of tfstat_search_host gets by default)
        for _ in range(3):
            pkg.tfstat_search_host(atoms_h, t_h, pkg.EXP, grid)
        t1 = time.perf_counter()
        for _ in range(3):
            pkg.tfstat_search_host(atoms_h, t_h, pkg.EXP, grid)
        ms_s_e2e = (time.perf_counter() - t1) / 3 * 1e3
        side["cfg4_exp_scan_e2e_host_buffers"] = {
            "ms_per_step": ms_s_e2e, "effective_terms_per_s": terms / (ms_s_e2e * 1e-3),
            "h2d_GBps": h2d / (ms_s_e2e * 1e-3) / 1e9}
        # roofline of the path a caller gets by default (EXP_AUTO = the sliding form): the weighted
        # terms the two kernels EXECUTED, counted by the kernels themselves (tfstat_opts.stats, in a
        # separate untimed call), as FP32 lane-ops, plus the fp32 closure + marginal update per
        # cell (23 lane-ops: csrc/exp_scan.cu)
        plan_s = pkg.plan_info(pkg.EXP, int(t.shape[0]), n_tpl, grid, exp_method=pkg.EXP_SCAN)
        st = torch.zeros(pkg.binding.N_STATS, dtype=torch.int64, device="cuda")
        pkg.tfstat_search(atoms, t, pkg.EXP, grid, exp_method=pkg.EXP_SCAN, stats=st)
        stv = dict(zip(pkg.binding.STAT_NAMES, (int(x) for x in st.cpu().numpy())))
        ev_s = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
        ev_s[0].record(), ev_s[1].record()
        pkg.tfstat_search(atoms, t, pkg.EXP, grid, workspace=ws_s, out=out_s,
                          exp_method=pkg.EXP_SCAN, main_kernel_events=ev_s)
        torch.cuda.synchronize()
        k_ms_s = ev_s[0].elapsed_time(ev_s[1])
        tpc = plan_s["tile_c"] % 10
        w_terms = (stv["terms_window"] + stv["terms_enter"] + stv["terms_leave"] +
                   stv["terms_resum"])
        # window sums (exp_window_kernel): the multiplicative recurrence, 7 multiply-adds per term
        # and nothing else; entering / leaving / re-summed atoms: 7 + 2 / TPC (weight argument, E^2)
        slide_terms = stv["terms_enter"] + stv["terms_leave"] + stv["terms_resum"]
        # grouped window sums (exp_moment_kernel): 7 multiply-adds per (atom, moment, template)
        # term + the 22 FP32 operations of a thread's four weights and their squares per atom,
        # shared by its 8 terms
        mom_terms = stv.get("terms_moment", 0)
        # the same search with EVERY window sum by the per-tau recurrence (tile code 1000): the
        # work the grouped sums stand for, for `frac_per_tau_form` below
        st.zero_()
        pkg.tfstat_search(atoms, t, pkg.EXP, grid, exp_method=pkg.EXP_SCAN, stats=st,
                          tile=(1000, 0, 0))
        stv_pt = dict(zip(pkg.binding.STAT_NAMES, (int(x) for x in st.cpu().numpy())))
        lane_ops_pt = (7.0 * (stv_pt["terms_window"] + slide_terms) + 2.0 * slide_terms / tpc +
                       23.0 * stv_pt["cells"])
        lane_ops = (7.0 * w_terms + 2.0 * slide_terms / tpc + 23.0 * stv["cells"] +
                    (7.0 + 22.0 / 8.0) * mom_terms)
        packed_b = plan_packed_bytes(int(t.shape[0]), n_tpl)
        side["cfg4_exp_scan_roofline"] = {
            "bound": "alu", "kernel": "exp_window_kernel + exp_moment_kernel + exp_slide_kernel",
            "kernel_ms": k_ms_s,
            "executed": stv, "weighted_terms": w_terms, "moment_terms": mom_terms,
            "templates_per_cta": tpc,
            "executed_fp32_lane_ops": lane_ops,
            "achieved": lane_ops / (k_ms_s * 1e-3) / 1e12, "peak": peak_ops / 1e12,
            "unit": "T FP32 lane-op/s", "frac": lane_ops / (k_ms_s * 1e-3) / peak_ops,
            "per_tau_form_fp32_lane_ops": lane_ops_pt,
            "frac_per_tau_form": lane_ops_pt / (k_ms_s * 1e-3) / peak_ops,
            "note": ("frac counts the EXECUTED lane-ops; the grouped window sums (8 moments per "
                     "group of 16-64 tau) execute fewer than the per-tau recurrence they replace, "
                     "whose lane-ops / this time / peak is frac_per_tau_form"),
            "hbm_floor_us": packed_b / (peaks["hbm_gbs"] * 1e9) * 1e6,
            "hbm_frac": packed_b / (k_ms_s * 1e-3) / 1e9 / peaks["hbm_gbs"],
            "terms_vs_direct": terms / max(w_terms + mom_terms, 1), "plan": plan_s}
        side["cfg4_exp_scan"] = {"ms_per_step": ms_s, "effective_terms_per_s": terms / (ms_s * 1e-3),
                                 "speedup_vs_direct": ms_per_step / ms_s,
                                 "max_rel_diff_max2F_vs_direct": dmax,
                                 "argmax_equal_frac": float(np.mean((r_s["m"] == r_d["m"]) &
                                                                    (r_s["n"] == r_d["n"])))}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD, "templates_per_gpu": n_tpl, "n_atoms": int(t.shape[0]),
                   "N_t0": grid.N_t0, "N_tau": grid.N_tau, "window": "exp",
                   "exp_method": "direct", "terms_per_step_per_gpu": terms,
                   "cells_per_step_per_gpu": cells,
                   "l2": f"inputs {atoms.numel() * 4 / 2**20:.0f} MiB per step > 126 MB L2, no flush",
                   "parallelism": f"templates sharded over {world} GPU(s), no collective"},
        "cells_per_s": cells * world / (ms_per_step * 1e-3),
        "e2e": {"value": terms * world / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3},
        "gpu_launches": plan["n_launches"] * args.steps,
        "roofline": roofline,
        "cpu_baseline": cpu,
        "clocks": clocks,
        "other_workloads": side,
    }
    print(json.dumps(line))
    if dist:
        dist.destroy_process_group()
    return 0


def run_leg(args):
    """One small workload, a few calls, for profiling (ncu -k ... python bench.py --leg ...): not a
    bench line."""
    import torch

    import paper_1805_05652_b200 as pkg
    from synth import make_workload
    from synth.atoms import Grid as SGrid, make_atoms

    torch.cuda.set_device(0)
    if args.leg == "exp_scan":  # config 4 through the default (sliding) form
        wl = make_workload(4, templates=list(range(args.templates)))
        a, t = torch.from_numpy(wl.data.atoms).cuda(), torch.from_numpy(wl.data.t).cuda()
        fn = lambda: pkg.tfstat_search(a, t, pkg.EXP, wl.grid)
    elif args.leg == "rect_1yr":  # one year at dt0 = dtau = T_SFT, rows 16-byte aligned
        n_y = 17520
        t_y = np.arange(n_y, dtype=np.int64) * 1800
        a = torch.from_numpy(make_atoms(t_y, np.random.default_rng(11)).astype(np.float32)).cuda()
        t = torch.from_numpy(t_y.astype(np.int32)).cuda()
        g_y = SGrid(0, 1800, n_y - 2, 3600, 1800, n_y - 4)
        m_y = torch.empty((g_y.N_t0, g_y.N_tau), dtype=torch.float32, device="cuda")
        fn = lambda: pkg.tfstat_map(a, t, pkg.RECT, g_y, out_map=m_y, rect_method=1)
    elif args.leg == "cfg5_rect":
        wl = make_workload(5)
        a, t = torch.from_numpy(wl.data.atoms[0]).cuda(), torch.from_numpy(wl.data.t).cuda()
        m5 = torch.empty((wl.grid.N_t0, wl.grid.N_tau), dtype=torch.float32, device="cuda")
        fn = lambda: pkg.tfstat_map(a, t, pkg.RECT, wl.grid, out_map=m5)
    else:
        raise SystemExit(f"unknown --leg {args.leg}")
    for _ in range(args.warmup):
        fn()
    ms = time_calls(torch, fn, args.steps)
    print(json.dumps({"leg": args.leg, "ms_per_call": ms, "calls": args.steps}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--templates", type=int, default=4096,
                    help="templates per GPU (4096 = BASELINE.json configs[3]; smaller values are "
                         "for debugging only and are not a valid bench line)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-side", action="store_true", help="skip the other-config numbers")
    ap.add_argument("--leg", default=None, choices=["exp_scan", "rect_1yr", "cfg5_rect"],
                    help="profiling aid: run ONE small workload a few times and exit")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.leg:
        return run_leg(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
