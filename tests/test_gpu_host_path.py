"""GPU parity of the END-TO-END entry point tfstat_search_host (host buffers in, host results out:
the paper's copy-in / kernel / copy-out per template, batched) against the fp64
oracle, through every kernel family and with ragged last chunks; plus the opt-in time-stamp
validator of include/tfstat.h (-m gpu)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from synth import Grid, tiny_workload  # noqa: E402
from tests.parity import check_cells, check_result  # noqa: E402

pytestmark = pytest.mark.gpu

RECT, EXP = 0, 1


@pytest.fixture(scope="module")
def pkg():
    import paper_1805_05652_b200 as p

    p.load_library()
    assert torch.cuda.is_available()
    return p


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def pinned(x):
    return torch.from_numpy(np.ascontiguousarray(x)).pin_memory()


def _chunk_budget(pkg, a_h, window, grid, tc, want_maps, **kw):
    """A device budget that makes tfstat_search_host settle on chunks of `tc` templates."""
    n = pkg.search_host_scratch_bytes(a_h.stride(0), a_h.shape[2], tc, window, grid,
                                      want_maps=want_maps, **kw)
    # results of ALL templates live in the scratch too; the helper above sized them for tc
    return n + 20 * a_h.shape[0] + 512


@pytest.mark.parametrize("want_maps", [True, False])
def test_host_path_lattice_rect_kernels_several_chunks(pkg, want_maps):
    """Rectangular window through the lattice kernels (bounds -> prefix/steps -> running sums),
    11 templates in chunks of 3 (+ a ragged 2): the chunks after the first reuse the bounds tables
    and take the cudaMemsetAsync branch for the scan flags.  Every template against the oracle."""
    grid = Grid(0, 1800, 40, 3600, 1800, 120)  # 4800 cells: too many for the one-launch kernel
    wl = tiny_workload(301, 300, 0.1, grid, n_templates=11, phi_random=True)
    a_h, t_h = pinned(wl.data.atoms), pinned(wl.data.t)
    assert pkg.plan_info(RECT, int(t_h.shape[0]), 3, grid)["kernel_name"] == "rect_run"
    budget = _chunk_budget(pkg, a_h, RECT, grid, 3, want_maps)
    res, maps = pkg.tfstat_search_host(a_h, t_h, RECT, grid, want_maps=want_maps,
                                       max_device_bytes=budget)
    for k in range(wl.n_templates):
        ref = oracle.map2F(wl.data.atoms[k], wl.data.t, RECT, grid)
        check_result(res[k], ref["twoF"], ref["flags"], grid.N_tau, f"host rect tpl{k}")
        if want_maps:
            check_cells(maps[k].numpy(), None, ref, f"host rect tpl{k}")
    # the same through the device-pointer call: identical bits
    r_dev = pkg.tfstat_search(dev(wl.data.atoms), dev(wl.data.t), RECT, grid)
    assert np.array_equal(res, r_dev.numpy())


def test_host_path_mixed_small_chunks_then_ragged_lattice_chunk(pkg):
    """n_templates = 2369: four chunks of 592 take the one-launch small-map kernel (which needs no
    bounds tables), the ragged last chunk of ONE template takes the lattice kernels and must
    build the tables itself.  All 2369 marginals against the oracle's batched search, maps of the
    first, a middle and the ragged template cell by cell."""
    grid = Grid(0, 1800, 100, 3600, 1800, 100)  # 10 000 cells
    T = 2369
    wl = tiny_workload(302, 600, 0.05, grid, n_templates=T, phi_random=True)
    n_atoms = int(wl.data.t.shape[0])
    assert n_atoms <= 2048
    assert pkg.plan_info(RECT, n_atoms, 592, grid)["kernel_name"] == "rect_small"
    assert pkg.plan_info(RECT, n_atoms, T % 592, grid)["kernel_name"] == "rect_run"
    a_h, t_h = pinned(wl.data.atoms), pinned(wl.data.t)
    res, maps = pkg.tfstat_search_host(a_h, t_h, RECT, grid, want_maps=True)
    ref, _ = oracle.search(wl.data.atoms, wl.data.t, RECT, grid)
    from tests.parity import TOL_2F, TOL_LOGB
    for k, mg in enumerate(ref):
        got = res[k]
        assert got["n_valid"] == mg.n_valid, f"tpl {k}"
        assert abs(got["max2F"] - mg.max2F) <= TOL_2F * max(1.0, mg.max2F), f"tpl {k}: max2F"
        assert abs(got["logB"] - mg.logB) <= TOL_LOGB * max(1.0, abs(mg.logB)), f"tpl {k}: logB"
        if (int(got["m"]), int(got["n"])) != (mg.m, mg.n):  # allowed only on a tie in the oracle
            full = oracle.map2F(wl.data.atoms[k], wl.data.t, RECT, grid)
            check_result(got, full["twoF"], full["flags"], grid.N_tau, f"tpl {k}")
    for k in (0, 1000, T - 1):
        full = oracle.map2F(wl.data.atoms[k], wl.data.t, RECT, grid)
        check_cells(maps[k].numpy(), None, full, f"host mixed tpl{k}")
        check_result(res[k], full["twoF"], full["flags"], grid.N_tau, f"host mixed tpl{k}")


@pytest.mark.parametrize("method", ["scan", "direct"])
def test_host_path_exp_ragged_chunk_needs_more_workspace(pkg, method):
    """Exponential window, 1000 templates = 3 chunks of 256 + a ragged 232.  The sliding form picks
    its tiles from the number of templates, so the ragged chunk's plan needs MORE workspace than a
    full chunk's: the scratch must be sized for both.  Host path == device path bit for bit, and
    templates of every chunk against the oracle."""
    grid = Grid(0, 1800, 1000, 3600, 1800, 64)
    T = 1000
    wl = tiny_workload(303, 400, 0.05, grid, n_templates=T, phi_random=True)
    n_atoms = int(wl.data.t.shape[0])
    em = pkg.EXP_SCAN if method == "scan" else pkg.EXP_DIRECT
    # (the plans of a 256-template chunk and of the 232-template remainder differ: tile shapes
    # follow the number of templates; whichever needs more, the scratch must hold both)
    full_plan = pkg.plan_info(EXP, n_atoms, 256, grid, exp_method=em)
    last_plan = pkg.plan_info(EXP, n_atoms, 232, grid, exp_method=em)
    assert full_plan["kernel"] == last_plan["kernel"]
    a_h, t_h = pinned(wl.data.atoms), pinned(wl.data.t)
    res, _ = pkg.tfstat_search_host(a_h, t_h, EXP, grid, exp_method=em)
    r_dev = pkg.tfstat_search(dev(wl.data.atoms), dev(wl.data.t), EXP, grid, exp_method=em).numpy()
    if method == "direct":
        assert np.array_equal(res, r_dev)  # per-template results do not depend on the batch
    else:  # two templates per CTA share the re-sum guard: last bits may depend on the neighbour
        assert np.array_equal(res["n_valid"], r_dev["n_valid"])
        assert np.allclose(res["max2F"], r_dev["max2F"], rtol=1e-4, atol=1e-4)
        assert np.allclose(res["logB"], r_dev["logB"], rtol=1e-4, atol=1e-4)
    for k in (0, 255, 256, 600, 767, 768, 900, T - 1):
        ref = oracle.map2F(wl.data.atoms[k], wl.data.t, EXP, grid)
        check_result(res[k], ref["twoF"], ref["flags"], grid.N_tau, f"host exp {method} tpl{k}")


def test_host_path_maps_through_lattice_rect_and_exp(pkg):
    """Maps copied back chunk by chunk (double-buffered device map buffers), rect and exp, with a
    ragged last chunk; every cell of every template against the oracle."""
    grid = Grid(-3600, 900, 70, 1800, 2700, 90)
    wl = tiny_workload(304, 500, 0.2, grid, n_templates=7, phi_random=True)
    a_h, t_h = pinned(wl.data.atoms), pinned(wl.data.t)
    for window, kw in ((RECT, {}), (EXP, {"exp_method": pkg.EXP_SCAN}),
                       (EXP, {"exp_method": pkg.EXP_DIRECT})):
        budget = _chunk_budget(pkg, a_h, window, grid, 2, True, **kw)
        res, maps = pkg.tfstat_search_host(a_h, t_h, window, grid, want_maps=True,
                                           max_device_bytes=budget, **kw)
        for k in range(wl.n_templates):
            ref = oracle.map2F(wl.data.atoms[k], wl.data.t, window, grid)
            check_cells(maps[k].numpy(), None, ref, f"host w{window} {kw} tpl{k}")
            check_result(res[k], ref["twoF"], ref["flags"], grid.N_tau, f"host w{window} {kw} tpl{k}")


def test_validate_timestamps(pkg):
    """The opt-in validator of the precondition 't_atoms strictly increasing' (gaps are fine)."""
    t = (np.arange(5000, dtype=np.int64) * 1800)
    t = np.delete(t, np.arange(100, 400))  # a gap is not a violation
    t = t.astype(np.int32)
    assert pkg.validate_timestamps(dev(t)) == -1
    assert pkg.validate_timestamps(dev(t[:1])) == -1
    dup = t.copy()
    dup[3000] = dup[2999]  # duplicate
    assert pkg.validate_timestamps(dev(dup)) == 3000
    uns = t.copy()
    uns[[10, 4000]] = uns[[4000, 10]]  # two swaps: the FIRST violation is reported
    assert pkg.validate_timestamps(dev(uns)) == 11
    uns2 = t.copy()
    uns2[-1] = 0
    assert pkg.validate_timestamps(dev(uns2)) == len(t) - 1


@pytest.mark.parametrize("cpt", [1, 2, 4])
def test_general_nan_atoms_only_spoil_their_own_windows(pkg, cpt):
    """tfstat_map_general with several tau cells per thread: an atom beyond a cell's own window
    must be skipped, not weighted by zero (0 x NaN), so a bad SFT spoils exactly the windows that
    hold it -- as in the oracle."""
    grid = Grid(0, 1800, 50, 3600, 1800, 600)
    wl = tiny_workload(305, 400, 0.0, grid)
    atoms, t = wl.data.atoms[0].copy(), wl.data.t
    atoms[:, 90] = np.nan
    atoms[4, 200] = np.inf
    for window, k in ((EXP, 3), (RECT, 1)):
        with np.errstate(invalid="ignore"):
            ref = oracle.map2F(atoms, t, window, grid)
        t0 = grid.t0()[:, None]
        tau = grid.tau()[None, :]
        hit = np.zeros((grid.N_t0, grid.N_tau), bool)
        for bad_t in (t[90], t[200]):
            hit |= (bad_t >= t0) & (bad_t < t0 + k * tau)
        assert hit.any() and (~hit).any()
        mg, fg, rg = pkg.tfstat_map_general(dev(atoms), dev(t), window, (k, 1),
                                            dev(grid.t0().astype(np.int32)),
                                            dev(grid.tau().astype(np.int32)), want_flags=True,
                                            cells_per_thread=cpt)
        mg, fg = mg.cpu().numpy(), fg.cpu().numpy()
        assert np.all(fg[hit] & 2) and np.all(mg[hit] == 0.0) and np.all(fg[~hit] == 0)
        err = np.abs(mg[~hit] - ref["twoF"][~hit])
        assert np.all(err <= 1e-3 * np.maximum(1.0, ref["twoF"][~hit]))
        assert rg.numpy()[0]["n_valid"] == int((~hit).sum())
