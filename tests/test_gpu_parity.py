"""GPU parity: the CUDA path through the C ABI against the fp64 oracle, element by element on
the same seeded inputs (-m gpu).  Sizes span several tiles and a ragged tail; the five
BASELINE.json configs are covered in full or on sampled cells the oracle computes one by one."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from synth import Grid, make_workload, tiny_workload  # noqa: E402
from tests.golden.load_golden import load  # noqa: E402
from tests.parity import TOL_2F, check_cells, check_result  # noqa: E402

pytestmark = pytest.mark.gpu

RECT, EXP = 0, 1


@pytest.fixture(scope="module")
def pkg():
    import paper_1805_05652_b200 as p

    p.load_library()  # fails loudly if libtfstat.so is missing: there is no fallback
    assert torch.cuda.is_available()
    return _DirectByDefault(p)


class _DirectByDefault:
    """The package with exp_method defaulting to EXP_DIRECT, so that every test written against
    the default exercises the direct-sum kernel; the sliding form (what EXP_AUTO resolves to) is
    tested by the tests that ask for EXP_SCAN / EXP_AUTO explicitly."""

    def __init__(self, p):
        self._p = p

    def __getattr__(self, name):
        f = getattr(self._p, name)
        if name in ("tfstat_map", "tfstat_search", "tfstat_search_host", "workspace_bytes",
                    "search_host_scratch_bytes"):
            def g(*a, **k):
                k.setdefault("exp_method", self._p.EXP_DIRECT)
                return f(*a, **k)
            return g
        return f


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def run_map(pkg, atoms, t, window, grid, **kw):
    m, f = pkg.tfstat_map(dev(atoms), dev(t), window, grid, want_flags=True, **kw)
    torch.cuda.synchronize()
    return m.cpu().numpy(), f.cpu().numpy()


# ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("wname,window", [("rect", RECT), ("exp", EXP)])
def test_T0_toy(pkg, wname, window):
    g = load("T0_toy.txt")
    atoms = np.stack([g[k] for k in ("a2", "b2", "ab", "FaRe", "FaIm", "FbRe", "FbIm")]).astype(
        np.float32)
    t = g["t_atoms"].astype(np.int32)
    grid = Grid(*(int(x) for x in g["grid_t0"]), *(int(x) for x in g["grid_tau"]))
    m, f = run_map(pkg, atoms, t, window, grid)
    np.testing.assert_allclose(m.ravel(), g[f"{wname}_2F"], rtol=2e-6, atol=2e-6)
    assert np.array_equal((f.ravel() != 0).astype(int), g[f"{wname}_flagged"].astype(int))
    r = pkg.tfstat_marginalise(dev(m), dev(f)).numpy()[0]
    assert r["m"] * grid.N_tau + r["n"] == int(g[f"{wname}_argmax_flat"][0])
    assert r["n_valid"] == int(g[f"{wname}_n_valid"][0])
    assert abs(r["logB"] - g[f"{wname}_logB"][0]) < 1e-5
    assert abs(r["max2F"] - g[f"{wname}_max2F"][0]) < 1e-5


TINY = [
    # seed, slots, gaps, grid                                    what it exercises
    (101, 64, 0.0, Grid(0, 1800, 12, 3600, 1800, 10)),          # smallest tile shape
    (102, 400, 0.2, Grid(0, 1800, 37, 3600, 1800, 300)),        # several n-blocks, ragged tails
    (103, 300, 0.3, Grid(-5400, 2700, 45, 1800, 3100, 150)),    # off-lattice steps, before data
    (104, 500, 0.1, Grid(400 * 1800, 900, 130, 7200, 7200, 70)),  # windows overrun the data end
    (105, 2500, 0.15, Grid(0, 1800, 50, 43200, 1800, 700)),     # > 1 staging chunk of atoms
    (106, 200, 0.1, Grid(0, 1801, 40, 3600, 1800, 1000)),       # gcd 1: per-cell binary search
    (107, 120, 0.0, Grid(0, 1800, 1, 3600, 1800, 90)),          # N_t0 = 1
    (108, 120, 0.0, Grid(0, 1800, 75, 7200, 1800, 1)),          # N_tau = 1
    (109, 1200, 0.1, Grid(0, 1801, 40, 3600, 4801, 900)),       # lattice > 2^22 points for rect too
]


@pytest.mark.parametrize("window", [RECT, EXP])
@pytest.mark.parametrize("seed,slots,gaps,grid", TINY)
def test_tiny_maps(pkg, window, seed, slots, gaps, grid):
    wl = tiny_workload(seed, slots, gaps, grid)
    atoms, t = wl.data.atoms[0], wl.data.t
    ref = oracle.map2F(atoms, t, window, grid)
    m, f = run_map(pkg, atoms, t, window, grid)
    check_cells(m, f, ref, f"tiny{seed}")
    assert pkg.count_terms(dev(t), window, grid) == int(ref["cnt"].sum())
    r = pkg.tfstat_marginalise(dev(m), dev(f)).numpy()[0]
    check_result(r, ref["twoF"], ref["flags"], grid.N_tau, f"tiny{seed} marginalise")
    if window == RECT:
        # both families of rectangular kernels on every case: 1 = lattice / per-cell kernels,
        # 2 = the one-launch small-map kernel (needs n_atoms <= 2048)
        for method in (1, 2) if t.shape[0] <= 2048 else (1,):
            m2, f2 = run_map(pkg, atoms, t, window, grid, rect_method=method)
            check_cells(m2, f2, ref, f"tiny{seed} rect_method {method}")
            res = pkg.tfstat_search(dev(atoms[None]), dev(t), window, grid, rect_method=method)
            check_result(res.numpy()[0], ref["twoF"], ref["flags"], grid.N_tau,
                         f"tiny{seed} rect_method {method} fused")


@pytest.mark.parametrize("window", [RECT, EXP])
def test_search_batched_small(pkg, window):
    """Batched fused search == per-template map + marginalise == oracle; padded layout."""
    grid = Grid(0, 1800, 23, 3600, 3600, 140)
    wl = tiny_workload(201, 350, 0.1, grid, n_templates=7, phi_random=True)
    T, _, N = wl.data.atoms.shape
    ld, tstride = N + 5, 7 * (N + 5) + 11  # padded rows and templates
    buf = torch.full((T * tstride,), float("nan"), dtype=torch.float32, device="cuda")
    a = torch.as_strided(buf, (T, 7, N), (tstride, ld, 1))
    a.copy_(dev(wl.data.atoms))
    res = pkg.tfstat_search(a, dev(wl.data.t), window, grid, want_maps=True, want_flags=True)
    torch.cuda.synchronize()
    got = res.numpy()
    for k in range(T):
        ref = oracle.map2F(wl.data.atoms[k], wl.data.t, window, grid)
        check_cells(res.maps[k].cpu().numpy(), res.flags[k].cpu().numpy(), ref, f"tpl{k}")
        check_result(got[k], ref["twoF"], ref["flags"], grid.N_tau, f"tpl{k}")
    # results-only call gives the same records
    res2 = pkg.tfstat_search(a, dev(wl.data.t), window, grid)
    assert np.array_equal(res2.numpy(), got)
    if window == RECT:  # the batched call through both families of rectangular kernels
        for method in (1, 2):
            r3 = pkg.tfstat_search(a, dev(wl.data.t), window, grid, want_maps=True,
                                   want_flags=True, rect_method=method)
            for k in range(T):
                ref = oracle.map2F(wl.data.atoms[k], wl.data.t, window, grid)
                check_cells(r3.maps[k].cpu().numpy(), r3.flags[k].cpu().numpy(), ref,
                            f"tpl{k} rect_method {method}")
                check_result(r3.numpy()[k], ref["twoF"], ref["flags"], grid.N_tau,
                             f"tpl{k} rect_method {method}")


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_search_equals_unsharded(pkg, world):
    """Template sharding (paper_1805_05652_b200/shard.py): every rank's contiguous shard run on
    its own gives bit-identical records to the one unsharded call (no data-path collective)."""
    grid = Grid(0, 1800, 23, 3600, 3600, 140)
    wl = tiny_workload(204, 300, 0.1, grid, n_templates=7, phi_random=True)
    a, t = dev(wl.data.atoms), dev(wl.data.t)
    for window in (EXP, RECT):
        full = pkg.tfstat_search(a, t, window, grid).numpy()
        parts = []
        for rank in range(world):
            lo, cnt = pkg.template_shard(a.shape[0], rank, world)
            if cnt:
                parts.append(pkg.tfstat_search(a[lo:lo + cnt], t, window, grid).numpy())
        assert np.array_equal(np.concatenate(parts), full)


@pytest.mark.parametrize("window,method", [(EXP, 0), (RECT, 1), (RECT, 2)])
def test_calls_are_capturable_in_a_cuda_graph(pkg, window, method):
    """The device-pointer calls only enqueue kernels on the caller's stream (no allocation, no
    synchronisation), so a search can be captured once and replayed on new atoms."""
    grid = Grid(0, 1800, 23, 3600, 3600, 140)
    wl = tiny_workload(205, 300, 0.0, grid, n_templates=3, phi_random=True)
    a, t = dev(wl.data.atoms), dev(wl.data.t)
    ws = torch.empty(pkg.workspace_bytes(window, int(t.shape[0]), 3, grid, rect_method=method),
                     dtype=torch.uint8, device="cuda")
    out = torch.empty((3, 5), dtype=torch.int32, device="cuda")
    call = lambda: pkg.tfstat_search(a, t, window, grid, workspace=ws, out=out,  # noqa: E731
                                     rect_method=method)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        call()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        call()
    for seed in (206, 207):  # replay on new atoms written into the captured buffers
        wl2 = tiny_workload(seed, 300, 0.0, grid, n_templates=3, phi_random=True)
        assert np.array_equal(wl2.data.t, wl.data.t)  # gapless: same time stamps
        a.copy_(dev(wl2.data.atoms))
        out.zero_()
        graph.replay()
        torch.cuda.synchronize()
        got = out.cpu().numpy().view(pkg.RESULT_DTYPE).reshape(-1)
        for k in range(3):
            ref = oracle.map2F(wl2.data.atoms[k], wl2.data.t, window, grid)
            check_result(got[k], ref["twoF"], ref["flags"], grid.N_tau, f"graph replay tpl{k}")
    # and the captured call itself reproduces the eager result
    a.copy_(dev(wl.data.atoms))
    eager = pkg.tfstat_search(a, t, window, grid, rect_method=method).numpy()
    graph.replay()
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy().view(pkg.RESULT_DTYPE).reshape(-1), eager)


@pytest.mark.parametrize("case", range(int(__import__("os").environ.get("TFSTAT_FUZZ_CASES", "64"))))
def test_random_grids_all_kernel_families(pkg, case):
    """Seeded random data sets and grids (odd steps, negative and late t0, tau from one second to
    longer than the data, heavy gaps, min_atoms 1..4) through every kernel family."""
    rng = np.random.default_rng(5000 + case)
    big = case % 8 == 7  # every eighth case: several staging chunks, CTAs and column tiles
    slots = int(rng.integers(20, 900)) * (6 if big else 1)
    gaps = float(rng.choice([0.0, 0.1, 0.4, 0.7]))
    dt0 = int(rng.choice([1800, 900, 2700, 1801, 3600, 7200, 777]))
    dtau = int(rng.choice([1800, 900, 3600, 5400, 1799, 43200, 1234]))
    N_t0, N_tau = int(rng.integers(1, 60)), int(rng.integers(1, 200))
    if big:
        N_t0, N_tau = 4 * N_t0, 3 * N_tau
    t0_min = int(rng.integers(-5, slots)) * 1800 + int(rng.choice([0, 0, 17]))
    tau_min = int(rng.choice([1, 1800, 3600, 1800 * 7 + 3]))
    grid = Grid(t0_min, dt0, N_t0, tau_min, dtau, N_tau)
    min_atoms = int(rng.integers(1, 5))
    T = 1 + case % 3  # the batched search sees 1..3 templates; maps are checked on the last one
    wl = tiny_workload(6000 + case, slots, gaps, grid, n_templates=T, phi_random=True)
    atoms, t = wl.data.atoms[T - 1], wl.data.t
    for window, kws in ((EXP, [{"exp_method": pkg.EXP_DIRECT}, {"exp_method": pkg.EXP_SCAN},
                                 {"exp_method": pkg.EXP_SCAN, "tile": (0, 0, 3)},
                                 {"exp_method": pkg.EXP_SCAN, "tile": (1000, 0, 0)}]),
                        (RECT, [{"rect_method": 1}, {"rect_method": 2},
                                  {"rect_method": 1, "tile": (2, 0, 0)},  # two rows per thread
                                  # seg_len < 0: the running-sum kernel where the tile kernel
                                  # would take over
                                  {"rect_method": 1, "tile": (0, 0, -1)},
                                  # the tile kernel (direct form) wherever the lattice qualifies
                                  {"rect_method": 1, "tile": (8, 0, 0)}])):
        ref = oracle.map2F(atoms, t, window, grid, min_atoms=min_atoms)
        for kw in kws:
            what = f"case {case} window {window} {kw}"
            m, f = run_map(pkg, atoms, t, window, grid, min_atoms=min_atoms, **kw)
            check_cells(m, f, ref, what)
            res = pkg.tfstat_search(dev(wl.data.atoms), dev(t), window, grid,
                                    min_atoms=min_atoms, **kw)
            check_result(res.numpy()[T - 1], ref["twoF"], ref["flags"], grid.N_tau, what)
        # the same window through the general entry point on arrays spelling out the grid
        mg, fg, rg = pkg.tfstat_map_general(dev(atoms), dev(t), window, (3, 1) if window == EXP else (1, 1),
                                            dev(grid.t0().astype(np.int32)),
                                            dev(grid.tau().astype(np.int32)), want_flags=True,
                                            min_atoms=min_atoms)
        check_cells(mg.cpu().numpy(), fg.cpu().numpy(), ref, f"case {case} window {window} general")
        check_result(rg.numpy()[0], ref["twoF"], ref["flags"], grid.N_tau,
                     f"case {case} window {window} general")
    # a random tabulated window with a rational support on the same (explicit) grid
    from oracle.binding import map2F_general

    sup = (int(rng.integers(1, 8)), int(rng.integers(1, 4)))
    table = rng.uniform(0.05, 1.0, size=int(rng.integers(2, 40))).astype(np.float32)
    t0g, taug = grid.t0().astype(np.int32), grid.tau().astype(np.int32)
    mg, fg, rg = pkg.tfstat_map_general(dev(atoms), dev(t), 2, sup, dev(t0g), dev(taug),
                                        table=dev(table), want_flags=True, min_atoms=min_atoms)
    reft = map2F_general(atoms, t, 2, sup, t0g, taug, table=table, min_atoms=min_atoms)
    check_cells(mg.cpu().numpy(), fg.cpu().numpy(), reft, f"case {case} table window")
    check_result(rg.numpy()[0], reft["twoF"], reft["flags"], grid.N_tau, f"case {case} table window")


def test_rect_maximum_grid_size_marginals(pkg):
    """The largest grid the ABI accepts (N_t0 N_tau just under 2^31 cells: flat indices up to the
    int32 limit), fused marginals only (the 8.6 GB map is never written).  n_valid is checked
    against integer window counts, the maximum against the oracle at the argmax and on a random
    sample, logB against its bounds."""
    N = 46340  # 46340^2 = 2 147 395 600 < 2^31
    grid = Grid(0, 1800, N, 1800, 1800, N)
    assert grid.n_cells < 2 ** 31 and (N + 1) ** 2 >= 2 ** 31
    lib = pkg.load_library()
    assert lib.tfstat_workspace_bytes(RECT, 100, 1, 0, 1800, N + 1, 1800, 1800, N + 1, None) == 0
    wl = tiny_workload(220, 60000, 0.1, grid)
    atoms, t = wl.data.atoms[0], wl.data.t
    res = pkg.tfstat_search(dev(atoms[None]), dev(t), RECT, grid).numpy()[0]
    # integer count of valid cells: cnt(m, n) >= 2, counts grow with n (all such cells have D > 0
    # here: two-detector atoms, checked on the sample below)
    t64 = t.astype(np.int64)
    lo = np.searchsorted(t64, grid.t0())
    n_valid = 0
    for m0 in range(0, N, 4096):  # rows in slabs: first n with >= 2 atoms in the window
        rows = slice(m0, min(m0 + 4096, N))
        need = np.minimum(lo[rows] + 1, len(t64) - 1)          # index of the window's 2nd atom
        has2 = lo[rows] + 1 < len(t64)
        tau_need = t64[need] - grid.t0()[rows] + 1              # smallest tau that includes it
        n_first = np.maximum(0, -(-(tau_need - grid.tau_min) // grid.dtau))
        n_valid += int(np.sum(np.where(has2, np.clip(N - n_first, 0, N), 0)))
    assert int(res["n_valid"]) == n_valid
    assert 0 <= res["m"] < N and 0 <= res["n"] < N
    at = oracle.cells(atoms, t, RECT, grid, np.array([res["m"]], np.int32),
                      np.array([res["n"]], np.int32))
    assert abs(at["twoF"][0] - res["max2F"]) <= TOL_2F * max(1.0, at["twoF"][0])
    rng = np.random.default_rng(3)
    ms = rng.integers(0, N, 3000).astype(np.int32)
    ns = rng.integers(0, N, 3000).astype(np.int32)
    smp = oracle.cells(atoms, t, RECT, grid, ms, ns)
    assert np.all(smp["twoF"] <= res["max2F"] * (1 + TOL_2F) + TOL_2F)
    assert np.all((smp["flags"] & 2) == ((smp["cnt"] == 0) * 2))  # D > 0 wherever there are atoms
    assert 0.5 * res["max2F"] - 1e-3 <= res["logB"] <= 0.5 * res["max2F"] + np.log(n_valid) + 1e-3


@pytest.mark.parametrize("scale", [1e-9, 1e-5, 1e6, 1e9])
def test_amplitude_scaling_far_from_unity(pkg, scale):
    """I5: (a2, b2, ab) x s^2 and (Fa, Fb) x s leave 2F unchanged.  With s = 1e9 the products
    A B overflow fp32, with s = 1e-9 they underflow: the fp32 fast paths must hand such cells to
    the fp64 closure instead of producing inf / NaN / 0."""
    grid = Grid(0, 1800, 40, 3600, 1800, 160)
    wl = tiny_workload(230, 500, 0.1, grid)
    atoms, t = wl.data.atoms[0], wl.data.t
    scaled = atoms.astype(np.float64).copy()
    scaled[0:3] *= scale * scale
    scaled[3:7] *= scale
    scaled = scaled.astype(np.float32)
    assert np.all(np.isfinite(scaled)) and np.all(scaled[0] > 0)
    for window, kws in ((EXP, [{"exp_method": pkg.EXP_DIRECT}, {"exp_method": pkg.EXP_SCAN}]),
                        (RECT, [{"rect_method": 1}, {"rect_method": 2}])):
        ref = oracle.map2F(scaled, t, window, grid)        # fp64: fine at any of these scales
        ref1 = oracle.map2F(atoms, t, window, grid)
        ok = ref1["flags"] == 0
        # I5 itself, up to the fresh fp32 rounding of the scaled atoms times the conditioning
        assert np.allclose(ref["twoF"][ok], ref1["twoF"][ok], rtol=2e-3, atol=2e-3)
        for kw in kws:
            m, f = run_map(pkg, scaled, t, window, grid, **kw)
            check_cells(m, f, ref, f"scale {scale} window {window} {kw}")
            res = pkg.tfstat_search(dev(scaled[None]), dev(t), window, grid, **kw)
            check_result(res.numpy()[0], ref["twoF"], ref["flags"], grid.N_tau,
                         f"scale {scale} window {window} {kw}")
    mg, fg, _ = pkg.tfstat_map_general(dev(scaled), dev(t), EXP, (3, 1),
                                       dev(grid.t0().astype(np.int32)),
                                       dev(grid.tau().astype(np.int32)), want_flags=True)
    check_cells(mg.cpu().numpy(), fg.cpu().numpy(), oracle.map2F(scaled, t, EXP, grid),
                f"scale {scale} general")


def test_nan_and_inf_atoms_only_spoil_their_own_windows(pkg):
    """A NaN atom and an inf atom (a bad SFT): every window that contains one is degenerate
    (flag bit 1, 2F = 0, out of the marginals), every other window is untouched -- also in the
    sliding form, where a bad atom that has LEFT the window must not linger in the running sums."""
    grid = Grid(0, 1800, 60, 3600, 1800, 40)
    wl = tiny_workload(240, 300, 0.0, grid)
    atoms, t = wl.data.atoms[0].copy(), wl.data.t
    atoms[:, 70] = np.nan
    atoms[3, 150] = np.inf
    for window, kws in ((EXP, [{"exp_method": pkg.EXP_DIRECT}, {"exp_method": pkg.EXP_SCAN},
                                 {"exp_method": pkg.EXP_SCAN, "tile": (0, 0, 7)}]),
                        (RECT, [{"rect_method": 1}, {"rect_method": 2}])):
        with np.errstate(invalid="ignore"):
            ref = oracle.map2F(atoms, t, window, grid)
        k = 3 if window == EXP else 1
        t0 = grid.t0()[:, None]
        tau = grid.tau()[None, :]
        hit = np.zeros((grid.N_t0, grid.N_tau), bool)
        for bad_t in (t[70], t[150]):
            hit |= (bad_t >= t0) & (bad_t < t0 + k * tau)
        assert hit.any() and (~hit).any()
        assert np.all(ref["flags"][hit] & 2) and np.all(ref["flags"][~hit] == 0)
        for kw in kws:
            what = f"window {window} {kw}"
            m, f = run_map(pkg, atoms, t, window, grid, **kw)
            assert np.all(f[hit] & 2) and np.all(m[hit] == 0.0), what
            assert np.all(f[~hit] == 0), what
            err = np.abs(m[~hit] - ref["twoF"][~hit])
            assert np.all(err <= TOL_2F * np.maximum(1.0, ref["twoF"][~hit])), what
            res = pkg.tfstat_search(dev(atoms[None]), dev(t), window, grid, **kw).numpy()[0]
            assert res["n_valid"] == int((~hit).sum()), what
            assert np.isfinite(res["max2F"]) and np.isfinite(res["logB"]), what
            assert abs(res["max2F"] - ref["twoF"][~hit].max()) <= TOL_2F * ref["twoF"][~hit].max()
        mg, fg, rg = pkg.tfstat_map_general(dev(atoms), dev(t), window, (k, 1),
                                            dev(grid.t0().astype(np.int32)),
                                            dev(grid.tau().astype(np.int32)), want_flags=True)
        mg, fg = mg.cpu().numpy(), fg.cpu().numpy()
        assert np.all(fg[hit] & 2) and np.all(mg[hit] == 0.0) and np.all(fg[~hit] == 0)
        assert np.all(np.abs(mg[~hit] - ref["twoF"][~hit]) <=
                      TOL_2F * np.maximum(1.0, ref["twoF"][~hit]))
        assert rg.numpy()[0]["n_valid"] == int((~hit).sum())


@pytest.mark.parametrize("case", range(24))
def test_marginalise_random_maps_with_ties(pkg, case):
    """tfstat_marginalise on random maps quantised so that the maximum is attained many times
    (the lowest flat index must win, exactly), with random flags, odd shapes (ragged tails,
    unaligned sizes), huge dynamic range in F, and all-flagged maps."""
    rng = np.random.default_rng(7000 + case)
    N_t0, N_tau = int(rng.integers(1, 400)), int(rng.integers(1, 700))
    levels = int(rng.choice([2, 5, 50, 100000]))
    scale = float(rng.choice([1.0, 30.0, 2000.0]))
    m = (rng.integers(0, levels, size=(N_t0, N_tau)) * (scale / levels)).astype(np.float32)
    p_flag = float(rng.choice([0.0, 0.1, 0.9, 1.0]))
    fl = (rng.random((N_t0, N_tau)) < p_flag).astype(np.uint8) * rng.integers(1, 4, (N_t0, N_tau)).astype(np.uint8)
    for flags in (None, fl):
        got = pkg.tfstat_marginalise(dev(m), None if flags is None else dev(flags)).numpy()[0]
        ref = oracle.marginalise(m.astype(np.float64), flags)
        assert got["n_valid"] == ref.n_valid
        if ref.n_valid == 0:
            assert (got["m"], got["n"], got["max2F"]) == (-1, -1, 0.0) and got["logB"] == -np.inf
            continue
        assert got["max2F"] == np.float32(ref.max2F)
        assert (got["m"], got["n"]) == (ref.m, ref.n)  # exact ties: lowest flat index
        assert abs(got["logB"] - ref.logB) <= 1e-4 * max(1.0, abs(ref.logB))


def test_concurrent_streams_do_not_interfere(pkg):
    """The library keeps no state between calls: searches enqueued on two streams at once, each
    with its own workspace, give the bits of the same searches run one after the other."""
    grid = Grid(0, 1800, 40, 3600, 1800, 260)
    wls = [tiny_workload(210 + i, 500, 0.1, grid, n_templates=5, phi_random=True) for i in (0, 1)]
    dat = [(dev(w.data.atoms), dev(w.data.t)) for w in wls]
    for window, kw in ((EXP, {}), (EXP, {"exp_method": pkg.EXP_SCAN}), (RECT, {"rect_method": 1})):
        ref = [pkg.tfstat_search(a, t, window, grid, **kw).numpy() for a, t in dat]
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        torch.cuda.synchronize()
        out = [None, None]
        for rep in range(4):  # interleave the enqueues
            for i in (0, 1):
                with torch.cuda.stream(streams[i]):
                    out[i] = pkg.tfstat_search(dat[i][0], dat[i][1], window, grid,
                                               stream=streams[i], **kw)
        torch.cuda.synchronize()
        for i in (0, 1):
            assert np.array_equal(out[i].numpy(), ref[i]), f"window {window} {kw}: stream {i}"


def test_search_host_equals_device(pkg):
    grid = Grid(0, 1800, 16, 3600, 1800, 100)
    wl = tiny_workload(202, 260, 0.05, grid, n_templates=9, phi_random=True)
    a_h = torch.from_numpy(wl.data.atoms).pin_memory()
    t_h = torch.from_numpy(wl.data.t).pin_memory()
    for window in (EXP, RECT):
        r_dev = pkg.tfstat_search(dev(wl.data.atoms), dev(wl.data.t), window, grid,
                                  want_maps=True)
        # small device budget (chunks of 2 of the 9 templates): several chunks go through the
        # double-buffered copies
        small = pkg.search_host_scratch_bytes(a_h.stride(0), a_h.shape[2], 2, window, grid,
                                              want_maps=True) + 256
        r_host, maps = pkg.tfstat_search_host(a_h, t_h, window, grid, want_maps=True,
                                              max_device_bytes=small)
        assert np.array_equal(r_host, r_dev.numpy())
        assert np.array_equal(maps.numpy(), r_dev.maps.cpu().numpy())
        # a scratch tensor of the caller, and the library's own cudaMalloc, give the same
        mine = torch.empty(small, dtype=torch.uint8, device="cuda")
        r2, maps2 = pkg.tfstat_search_host(a_h, t_h, window, grid, want_maps=True, scratch=mine)
        r3, maps3 = pkg.tfstat_search_host(a_h, t_h, window, grid, want_maps=True,
                                           library_malloc=True, max_device_bytes=small)
        r4, _ = pkg.tfstat_search_host(a_h, t_h, window, grid)  # cached scratch, results only
        for r, m in ((r2, maps2), (r3, maps3), (r4, None)):
            assert np.array_equal(r, r_dev.numpy())
            if m is not None:
                assert np.array_equal(m.numpy(), r_dev.maps.cpu().numpy())
        # a scratch too small for one template is an error, not a crash
        with pytest.raises(pkg.TfstatError):
            pkg.tfstat_search_host(a_h, t_h, window, grid, want_maps=True,
                                   scratch=torch.empty(4096, dtype=torch.uint8, device="cuda"))


def test_degenerate_maps(pkg):
    t = (np.arange(40) * 1800).astype(np.int32)
    wl = tiny_workload(203, 40, 0.0, Grid(0, 1800, 2, 3600, 1800, 2))
    atoms = wl.data.atoms[0]
    for window in (RECT, EXP):
        # every window lies after the data: all cells empty, not an error
        g = Grid(10 ** 6, 1800, 5, 3600, 1800, 40)
        res = pkg.tfstat_search(dev(atoms[None]), dev(t), window, g, want_maps=True,
                                want_flags=True)
        r = res.numpy()[0]
        assert (r["n_valid"], r["m"], r["n"], r["max2F"]) == (0, -1, -1, 0.0)
        assert r["logB"] == -np.inf
        assert torch.all(res.maps == 0) and torch.all(res.flags == 3)
        # min_atoms is honoured
        g2 = Grid(0, 1800, 6, 1800, 1800, 5)
        for min_atoms in (1, 2, 4):
            ref = oracle.map2F(atoms, t, window, g2, min_atoms=min_atoms)
            m, f = run_map(pkg, atoms, t, window, g2, min_atoms=min_atoms)
            check_cells(m, f, ref, f"min_atoms={min_atoms}")
    # a single atom, single cell
    m, f = run_map(pkg, atoms[:, :1].copy(), t[:1], RECT, Grid(0, 1, 1, 1800, 1, 1))
    assert m[0, 0] == 0 and f[0, 0] & 1


# ---------------------------------------------------------------------------------------
# BASELINE.json configs
# ---------------------------------------------------------------------------------------
def test_config1_rect_full(pkg):
    wl = make_workload(1)
    atoms, t = wl.data.atoms[0], wl.data.t
    ref = oracle.map2F(atoms, t, RECT, wl.grid)
    m, f = run_map(pkg, atoms, t, RECT, wl.grid)
    check_cells(m, f, ref, "cfg1")
    assert np.count_nonzero(f) == 24
    r = pkg.tfstat_marginalise(dev(m), dev(f)).numpy()[0]
    check_result(r, ref["twoF"], ref["flags"], wl.grid.N_tau, "cfg1")


def test_config2_exp_full_map_and_injection(pkg):
    wl = make_workload(2)
    atoms, t = wl.data.atoms[0], wl.data.t
    ref = oracle.map2F(atoms, t, EXP, wl.grid)
    m, f = run_map(pkg, atoms, t, EXP, wl.grid)
    worst = check_cells(m, f, ref, "cfg2")
    assert worst < 0.5  # comfortably inside the tolerance, not just scraping it
    res = pkg.tfstat_search(dev(atoms[None]), dev(t), EXP, wl.grid)
    check_result(res.numpy()[0], ref["twoF"], ref["flags"], wl.grid.N_tau, "cfg2")
    (m_inj, n_inj, rho), = wl.injections.values()
    assert abs(int(res.numpy()[0]["m"]) - m_inj) <= 6
    assert pkg.count_terms(dev(t), EXP, wl.grid) == 436248960  # eq. (A.6)


def _sample_cells(grid, n, seed):
    rng = np.random.default_rng(seed)
    ms = rng.integers(0, grid.N_t0, size=n)
    ns = rng.integers(0, grid.N_tau, size=n)
    # always include the corners and the first/last rows and columns' ends
    ms[:4] = [0, 0, grid.N_t0 - 1, grid.N_t0 - 1]
    ns[:4] = [0, grid.N_tau - 1, 0, grid.N_tau - 1]
    return ms.astype(np.int32), ns.astype(np.int32)


@pytest.mark.parametrize("window", [EXP, RECT])
def test_config3_glitch_scale(pkg, window):
    wl = make_workload(3)
    atoms, t = wl.data.atoms[0], wl.data.t
    assert t.shape[0] == 4608
    m, f = run_map(pkg, atoms, t, window, wl.grid)
    if window == RECT:
        ref = oracle.map2F(atoms, t, window, wl.grid)
        check_cells(m, f, ref, "cfg3 rect")
        res = pkg.tfstat_search(dev(atoms[None]), dev(t), window, wl.grid)
        check_result(res.numpy()[0], ref["twoF"], ref["flags"], wl.grid.N_tau, "cfg3 rect")
    else:
        # the oracle's FULL map (2.1e9 window-atom terms: a few seconds on the host cores)
        ref = oracle.map2F(atoms, t, window, wl.grid)
        worst = check_cells(m, f, ref, "cfg3 exp")
        assert worst < 0.5
        res = pkg.tfstat_search(dev(atoms[None]), dev(t), window, wl.grid).numpy()[0]
        check_result(res, ref["twoF"], ref["flags"], wl.grid.N_tau, "cfg3 exp")


def _check_fused_equals_own_map(res, m, f, grid):
    """A property that holds at any size, checked IN ADDITION to the oracle: the fused marginals
    of a launch equal the fp64 marginals of the map the same launch wrote."""
    mg = oracle.marginalise(m.astype(np.float64), f)
    assert int(res["n_valid"]) == mg.n_valid
    assert abs(res["max2F"] - mg.max2F) <= 1e-6 * max(1.0, mg.max2F)
    assert (int(res["m"]), int(res["n"])) == (mg.m, mg.n)
    assert abs(res["logB"] - mg.logB) <= 1e-4 * max(1.0, abs(mg.logB))


_GOLDEN = {}


def _check_against_stored_oracle_marginals(res, name, wl, window, k=0):
    """res: one tfstat_result of template k; name: a file written by tests/golden/make_marginals.py
    (the oracle's marginals of the FULL fp64 map, too slow to recompute in every test run)."""
    from synth.atoms import BASE_SEED
    g = _GOLDEN.get(name) or _GOLDEN.setdefault(name, load(name))
    assert int(g["seed"][0]) == BASE_SEED + wl.config_id, "stored marginals are of another workload"
    max2F, logB = float(g["max2F"][k]), float(g["logB"][k])
    what = f"{name} tpl{k}"
    assert int(res["n_valid"]) == int(g["n_valid"][k]), what
    assert abs(res["max2F"] - max2F) <= TOL_2F * max(1.0, max2F), f"{what}: max2F"
    assert abs(res["logB"] - logB) <= 1e-4 * max(1.0, abs(logB)), f"{what}: logB"
    if (int(res["m"]), int(res["n"])) != (int(g["m"][k]), int(g["n"][k])):
        # another argmax is right only if the oracle's value THERE ties with its maximum
        at = oracle.cells(wl.data.atoms[k], wl.data.t, window, wl.grid,
                          np.array([res["m"]], np.int32), np.array([res["n"]], np.int32))
        assert at["flags"][0] == 0 and max2F - at["twoF"][0] <= TOL_2F * max(1.0, max2F), (
            f"{what}: argmax ({res['m']},{res['n']}) vs ({int(g['m'][k])},{int(g['n'][k])}) "
            "is not a tie")
        if "runner_up" in g:
            assert max2F - float(g["runner_up"][k]) <= TOL_2F * max(1.0, max2F)


def test_config4_batched_search_subset(pkg):
    """8 templates of config 4 (2 with injections), full oracle maps."""
    from synth.configs import cfg4_injection_plan

    plan = cfg4_injection_plan()
    inj = sorted(plan)[:2]
    idx = sorted(set([0, 1, 2, 3, 4, 5] + inj))
    wl = make_workload(4, templates=idx)
    res = pkg.tfstat_search(dev(wl.data.atoms), dev(wl.data.t), EXP, wl.grid).numpy()
    for j, k in enumerate(idx):
        ref = oracle.map2F(wl.data.atoms[j], wl.data.t, EXP, wl.grid)
        check_result(res[j], ref["twoF"], ref["flags"], wl.grid.N_tau, f"cfg4 tpl{k}")
        if k in plan:
            m_inj, n_inj, rho = plan[k]
            assert res[j]["max2F"] >= ref["twoF"][m_inj, n_inj] * (1 - 2 * TOL_2F)
            assert res[j]["max2F"] > 30.0  # rho = 8 stands out of chi^2_4 noise


def test_config4_full_launch_all_injected_templates(pkg):
    """BASELINE.json config 4 at full size, in the launch configuration bench.py times (one
    tfstat_search over all 4096 templates): the 41 injected templates and 7 noise-only ones are
    checked against the oracle's marginals (its full map where the argmax differs), every
    template's record is sane, and a sub-launch gives bit-identical records."""
    from synth.configs import cfg4_injection_plan

    plan = cfg4_injection_plan()
    wl = make_workload(4)
    assert wl.data.atoms.shape == (4096, 7, 2880) and len(plan) == 41
    a, t = dev(wl.data.atoms), dev(wl.data.t)
    res = pkg.tfstat_search(a, t, EXP, wl.grid).numpy()
    idx = sorted(plan) + [0, 1, 2, 1000, 2047, 3000, 4095]
    ref, _ = oracle.search(wl.data.atoms[idx], wl.data.t, EXP, wl.grid)
    for k, mg in zip(idx, ref):
        got = res[k]
        assert got["n_valid"] == mg.n_valid
        assert abs(got["max2F"] - mg.max2F) <= TOL_2F * max(1.0, mg.max2F), f"tpl {k}: max2F"
        assert abs(got["logB"] - mg.logB) <= 1e-4 * max(1.0, abs(mg.logB)), f"tpl {k}: logB"
        if (int(got["m"]), int(got["n"])) != (mg.m, mg.n):  # allowed only on a tie in the oracle
            full = oracle.map2F(wl.data.atoms[k], wl.data.t, EXP, wl.grid)
            check_result(got, full["twoF"], full["flags"], wl.grid.N_tau, f"cfg4 tpl{k}")
        if k in plan:
            assert got["max2F"] > 30.0  # rho = 8 stands out of chi^2_4 noise
    # ALL 4096 templates against the oracle's stored marginals (tests/golden/make_marginals.py:
    # 1.08e12 window-atom terms in fp64, computed once)
    for k in range(4096):
        _check_against_stored_oracle_marginals(res[k], "cfg4_exp_marginals.txt", wl, EXP, k)
    # every record: all cells valid (gapless data, tau >= 0.5 d), indices inside the grid,
    # maxF <= logB <= maxF + log(n_valid)
    assert np.all(res["n_valid"] == wl.grid.n_cells)
    assert np.all((res["m"] >= 0) & (res["m"] < wl.grid.N_t0) & (res["n"] >= 0) &
                  (res["n"] < wl.grid.N_tau))
    assert np.all(res["logB"] >= 0.5 * res["max2F"] - 1e-3)
    assert np.all(res["logB"] <= 0.5 * res["max2F"] + np.log(wl.grid.n_cells) + 1e-3)
    # templates are independent: a launch over a slice gives the same bits
    sub = pkg.tfstat_search(a[1000:1100], t, EXP, wl.grid).numpy()
    assert np.array_equal(sub, res[1000:1100])
    # and so does the exact sliding form, within tolerance, on all 4096
    scan = pkg.tfstat_search(a, t, EXP, wl.grid, exp_method=pkg.EXP_SCAN).numpy()
    for k in range(4096):
        _check_against_stored_oracle_marginals(scan[k], "cfg4_exp_marginals.txt", wl, EXP, k)


@pytest.mark.parametrize("window", [RECT, EXP])
def test_config5_year_sampled(pkg, window):
    wl = make_workload(5)
    atoms, t = wl.data.atoms[0], wl.data.t
    assert t.shape[0] == 13140
    res = pkg.tfstat_search(dev(atoms[None]), dev(t), window, wl.grid, want_maps=True,
                            want_flags=True)
    torch.cuda.synchronize()
    m, f = res.maps[0].cpu().numpy(), res.flags[0].cpu().numpy()
    ms, ns = _sample_cells(wl.grid, 20000 if window == EXP else 100000, 5)
    ref = oracle.cells(atoms, t, window, wl.grid, ms, ns)
    check_cells(m[ms, ns], f[ms, ns], ref, f"cfg5 w{window} sampled")
    # marginals against the oracle's FULL fp64 map (stored: tests/golden/make_marginals.py)
    _check_against_stored_oracle_marginals(
        res.numpy()[0], "cfg5_rect_marginals.txt" if window == RECT else "cfg5_exp_marginals.txt",
        wl, window)
    _check_fused_equals_own_map(res.numpy()[0], m, f, wl.grid)
    # the results-only launch (no map written: what a search uses) gives the same record
    res2 = pkg.tfstat_search(dev(atoms[None]), dev(t), window, wl.grid).numpy()[0]
    _check_against_stored_oracle_marginals(
        res2, "cfg5_rect_marginals.txt" if window == RECT else "cfg5_exp_marginals.txt", wl, window)
    # all cells the oracle says are count-degenerate on the last rows (end of data) are flagged
    last = oracle.cells(atoms, t, window, wl.grid, np.full(720, wl.grid.N_t0 - 1, np.int32),
                        np.arange(720, dtype=np.int32))
    assert np.array_equal(f[-1] & 1, last["flags"] & 1)


@pytest.mark.parametrize("n_tau", [17519, 17516])
def test_one_year_full_resolution_rect_map_sampled(pkg, n_tau):
    """The largest of the paper's setups (one year at dt0 = dtau = T_SFT,
    3.07e8 cells, 1.23 GB), in the launch configuration bench.py's rect_map_1yr_full_resolution
    leg times: rect_tile_kernel, 128 x 256-cell tiles.  N_tau = 17519 leaves the rows unaligned to
    16 bytes, 17516 aligns them (the running-sum kernel of round 1 cared; the tile kernel stores
    128-byte warp rows either way)."""
    from synth.atoms import Grid, make_atoms
    rng = np.random.default_rng(2026)
    t = np.arange(17520, dtype=np.int64) * 1800
    t = t[rng.random(t.shape[0]) > 0.01]  # 1 % of the SFTs missing
    atoms = make_atoms(t, rng).astype(np.float32)
    t = t.astype(np.int32)
    grid = Grid(0, 1800, 17518, 3600, 1800, n_tau)
    a_d, t_d = dev(atoms[None]), dev(t)
    m_d = torch.empty((grid.N_t0, grid.N_tau), dtype=torch.float32, device="cuda")
    pkg.tfstat_map(a_d[0], t_d, RECT, grid, out_map=m_d, rect_method=1)
    ms, ns = _sample_cells(grid, 60000, 17)
    # the end of the data: the last rows, whose windows run out of atoms
    ms[4:2004] = grid.N_t0 - 1 - (np.arange(2000) % 50)
    mi, ni = torch.from_numpy(ms.astype(np.int64)).cuda(), torch.from_numpy(ns.astype(np.int64)).cuda()
    got = m_d[mi, ni].cpu().numpy()
    res = pkg.tfstat_search(a_d, t_d, RECT, grid, want_maps=True, want_flags=True, rect_method=1)
    torch.cuda.synchronize()
    # the flag-writing launch computes the same cells bit for bit
    assert torch.equal(res.maps[0], m_d)
    f = res.flags[0][mi, ni].cpu().numpy()
    ref = oracle.cells(atoms, t, RECT, grid, ms, ns)
    check_cells(got, f, ref, f"one-year rect N_tau={n_tau} sampled")
    # fused marginals of the same launch against a GPU reduction of its own map
    r0 = res.numpy()[0]
    valid = res.flags[0] == 0
    assert int(r0["n_valid"]) == int(valid.sum().item())
    best = torch.where(valid, res.maps[0], torch.full_like(res.maps[0], -1.0)).max().item()
    assert float(r0["max2F"]) == best
    assert float(res.maps[0][int(r0["m"]), int(r0["n"])].item()) == best
    # ... and the oracle agrees on the value at that argmax
    at = oracle.cells(atoms, t, RECT, grid, np.array([r0["m"]], np.int32),
                      np.array([r0["n"]], np.int32))
    assert at["flags"][0] == 0 and abs(at["twoF"][0] - best) <= TOL_2F * max(1.0, at["twoF"][0])


TILE_GRIDS = [
    # slots, gaps, grid                                   lattice (e_m, e_n), what it exercises
    (700, 0.0, Grid(0, 1800, 300, 1800, 1800, 600)),       # (1, 1): 3 x 3 tiles, ragged both ways
    (700, 0.3, Grid(-3600, 1800, 200, 1, 1800, 300)),      # (1, 1): gaps, tau from one second, t0 before the data
    (900, 0.1, Grid(0, 900, 260, 3600, 1800, 280)),        # (1, 2): pairs two rows down, one column back
    (900, 0.1, Grid(0, 3600, 140, 1800, 900, 520)),        # (4, 1)
    (600, 0.2, Grid(300 * 1800, 1800, 150, 5400, 900, 300)),  # (2, 1): windows overrun the data
    (400, 0.0, Grid(0, 1800, 9, 3600, 3600, 40)),          # (1, 2): fewer rows than one pair group
]


@pytest.mark.parametrize("slots,gaps,grid", TILE_GRIDS)
def test_rect_tile_kernel_small_grids(pkg, slots, gaps, grid):
    """rect_tile_kernel (the direct, anchored form the one-year map runs through) forced on small
    grids (tile_c = 8; the plan itself only takes it when the map fills the GPU): every cell and
    flag of every template against the oracle, map + flags, map only and results only, with
    min_atoms 1..3 and a bad SFT."""
    T = 3
    wl = tiny_workload(7000 + slots + grid.N_t0, slots, gaps, grid, n_templates=T, phi_random=True)
    atoms, t = wl.data.atoms.copy(), wl.data.t
    atoms[1, :, len(t) // 3] = np.nan  # template 1: one bad SFT (every channel, R19)
    kw = {"rect_method": 1, "tile": (8, 0, 0)}
    assert pkg.plan_info(RECT, len(t), T, grid, **kw)["kernel_name"] == "rect_tile"
    assert pkg.plan_info(RECT, len(t), T, grid, rect_method=1)["kernel_name"] != "rect_tile"
    for min_atoms in (2, 1, 3):
        full = pkg.tfstat_search(dev(atoms), dev(t), RECT, grid, want_maps=True, want_flags=True,
                                 min_atoms=min_atoms, **kw)
        maps_only = pkg.tfstat_search(dev(atoms), dev(t), RECT, grid, want_maps=True,
                                      min_atoms=min_atoms, **kw)
        res_only = pkg.tfstat_search(dev(atoms), dev(t), RECT, grid, min_atoms=min_atoms, **kw)
        torch.cuda.synchronize()
        assert torch.equal(full.maps, maps_only.maps)
        assert np.array_equal(full.numpy(), maps_only.numpy())
        assert np.array_equal(full.numpy(), res_only.numpy())
        for k in range(T):
            with np.errstate(invalid="ignore"):
                ref = oracle.map2F(atoms[k], t, RECT, grid, min_atoms=min_atoms)
            what = f"rect tile {grid} min_atoms {min_atoms} tpl{k}"
            check_cells(full.maps[k].cpu().numpy(), full.flags[k].cpu().numpy(), ref, what)
            check_result(full.numpy()[k], ref["twoF"], ref["flags"], grid.N_tau, what)
    # the same bits through tfstat_map (one template, no batch)
    m, f = run_map(pkg, atoms[0], t, RECT, grid, min_atoms=3, **kw)
    assert np.array_equal(m, full.maps[0].cpu().numpy()) and np.array_equal(f, full.flags[0].cpu().numpy())


# ---------------------------------------------------------------------------------------
# exact factorised / sliding exponential path (SURVEY.md 8(a) row a3', TFSTAT_EXP_SCAN):
# the same oracle, the same tolerances
# ---------------------------------------------------------------------------------------
SCAN = 2


@pytest.mark.parametrize("seg_len", [0, 1, 7, 32])
@pytest.mark.parametrize("seed,slots,gaps,grid", TINY)
def test_tiny_maps_exp_scan(pkg, seed, slots, gaps, grid, seg_len):
    wl = tiny_workload(seed, slots, gaps, grid)
    atoms, t = wl.data.atoms[0], wl.data.t
    ref = oracle.map2F(atoms, t, EXP, grid)
    m, f = run_map(pkg, atoms, t, EXP, grid, exp_method=SCAN, tile=(0, 0, seg_len))
    check_cells(m, f, ref, f"scan tiny{seed} seg{seg_len}")
    res = pkg.tfstat_search(dev(atoms[None]), dev(t), EXP, grid, exp_method=SCAN,
                            tile=(0, 0, seg_len)).numpy()[0]
    check_result(res, ref["twoF"], ref["flags"], grid.N_tau, f"scan tiny{seed} seg{seg_len}")


def test_exp_auto_is_the_sliding_form(pkg):
    """EXP_AUTO (what a caller gets without options) resolves to the exact sliding form: same bits
    as EXP_SCAN, within tolerance of the oracle, and of the direct sum."""
    grid = Grid(0, 1800, 37, 3600, 1800, 300)
    wl = tiny_workload(102, 400, 0.2, grid, n_templates=3, phi_random=True)
    a, t = dev(wl.data.atoms), dev(wl.data.t)
    auto = pkg.tfstat_search(a, t, EXP, grid, exp_method=pkg.EXP_AUTO, want_maps=True,
                             want_flags=True)
    scan = pkg.tfstat_search(a, t, EXP, grid, exp_method=pkg.EXP_SCAN, want_maps=True,
                             want_flags=True)
    direct = pkg.tfstat_search(a, t, EXP, grid, exp_method=pkg.EXP_DIRECT, want_maps=True)
    assert np.array_equal(auto.numpy(), scan.numpy())
    assert torch.equal(auto.maps, scan.maps) and torch.equal(auto.flags, scan.flags)
    assert not torch.equal(auto.maps, direct.maps)  # a different kernel did run
    for k in range(3):
        ref = oracle.map2F(wl.data.atoms[k], wl.data.t, EXP, grid)
        check_cells(auto.maps[k].cpu().numpy(), auto.flags[k].cpu().numpy(), ref, f"auto tpl{k}")
        check_result(auto.numpy()[k], ref["twoF"], ref["flags"], grid.N_tau, f"auto tpl{k}")
    # NULL options at the C level are AUTO too
    lib = pkg.load_library()
    out = torch.empty((3, 5), dtype=torch.int32, device="cuda")
    ws = torch.empty(pkg.workspace_bytes(EXP, int(t.shape[0]), 3, grid, exp_method=pkg.EXP_AUTO),
                     dtype=torch.uint8, device="cuda")
    rc = lib.tfstat_search(a.data_ptr(), a.stride(0), a.stride(1), t.data_ptr(), int(t.shape[0]), 3,
                           EXP, grid.t0_min, grid.dt0, grid.N_t0, grid.tau_min, grid.dtau,
                           grid.N_tau, out.data_ptr(), None, None, ws.data_ptr(), ws.numel(),
                           torch.cuda.current_stream().cuda_stream, None)
    assert rc == 0
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy().view(pkg.RESULT_DTYPE).reshape(-1), auto.numpy())


def test_exp_scan_long_gaps_and_disjoint_windows(pkg):
    """Windows that lose most of their atoms while sliding (long gaps), windows shorter than
    the t0 step (no overlap between neighbours), tau >> data span, min_atoms variants."""
    rng = np.random.default_rng(77)
    slots = np.concatenate([np.arange(0, 40), np.arange(400, 420), np.arange(1000, 1300),
                            np.arange(1302, 1304), np.arange(2500, 2600)])
    t = (slots * 1800).astype(np.int32)
    from synth import make_atoms
    atoms = make_atoms(t, rng).astype(np.float32)
    for grid in (Grid(0, 1800, 700, 3600, 5400, 60),          # slides through the long gaps
                 Grid(0, 36000, 120, 1800, 1800, 12),          # 3 tau < dt0 for small tau: disjoint
                 Grid(-90000, 1800, 300, 86400 * 50, 86400 * 25, 40),  # tau >> span, starts before data
                 Grid(1000 * 1800, 900, 640, 1800, 900, 33)):  # half-slot steps
        ref = oracle.map2F(atoms, t, EXP, grid)
        for seg_len in (0, 50):
            m, f = run_map(pkg, atoms, t, EXP, grid, exp_method=SCAN, tile=(0, 0, seg_len))
            check_cells(m, f, ref, f"scan gaps {grid} seg{seg_len}")
    g = Grid(0, 1800, 50, 1800, 1800, 20)
    for min_atoms in (1, 3):
        ref = oracle.map2F(atoms, t, EXP, g, min_atoms=min_atoms)
        m, f = run_map(pkg, atoms, t, EXP, g, exp_method=SCAN, min_atoms=min_atoms)
        check_cells(m, f, ref, f"scan min_atoms={min_atoms}")


@pytest.mark.parametrize("tpc,seg_len", [(0, 0), (1, 0), (2, 5), (422, 0), (211, 7), (122, 3),
                                         (1000, 0), (1412, 4), (4, 0), (424, 3)])
def test_exp_scan_batched_equals_oracle_and_direct(pkg, tpc, seg_len):
    """7 templates: with 2 templates per CTA (shared weights) the last group is ragged; tpc also
    selects the tile of the window-sum kernel (10 x (10 RT + TPC): 4, 2 or 1 tau per thread)."""
    grid = Grid(0, 1800, 23, 3600, 3600, 140)
    wl = tiny_workload(201, 350, 0.1, grid, n_templates=7, phi_random=True)
    a, t = dev(wl.data.atoms), dev(wl.data.t)
    # (4 templates per CTA exist for 128-thread CTAs only: ask for them)
    tile = (tpc, 128 if tpc % 10 == 4 else 0, seg_len)
    if tpc % 10 == 4:
        assert pkg.plan_info(EXP, int(t.shape[0]), 7, grid, exp_method=SCAN, tile=tile)["tile_c"] % 10 == 4
    res = pkg.tfstat_search(a, t, EXP, grid, exp_method=SCAN, want_maps=True, want_flags=True,
                            tile=tile)
    direct = pkg.tfstat_search(a, t, EXP, grid, exp_method=1, want_flags=True)
    torch.cuda.synchronize()
    assert torch.equal(res.flags, direct.flags)
    got = res.numpy()
    for k in range(wl.n_templates):
        ref = oracle.map2F(wl.data.atoms[k], wl.data.t, EXP, grid)
        check_cells(res.maps[k].cpu().numpy(), res.flags[k].cpu().numpy(), ref, f"scan tpl{k}")
        check_result(got[k], ref["twoF"], ref["flags"], grid.N_tau, f"scan tpl{k}")


MOMENT_GRIDS = [
    # slots, gaps, grid, seg_len                            which tau regions the plan groups
    (2400, 0.0, Grid(0, 1800, 20, 1800, 1800, 700), 0),     # 32s above tau = 273 steps, 64s above 556
    (2400, 0.15, Grid(-7200, 1800, 33, 3600, 1800, 650), 7),  # gaps, t0 before the data, 5 segments
    (1500, 0.1, Grid(0, 3600, 12, 7200, 3600, 420), 0),     # dtau = 2 SFTs: windows overrun the data
    (1300, 0.3, Grid(0, 900, 40, 900, 900, 620), 16),       # half-SFT steps, heavy gaps
]


@pytest.mark.parametrize("slots,gaps,grid,seg_len", MOMENT_GRIDS)
def test_exp_scan_grouped_window_sums(pkg, slots, gaps, grid, seg_len):
    """exp_moment_kernel: the window sums of large tau in groups of 32 / 64 neighbouring tau by the
    Taylor expansion in 1/tau.  Grids on which the plan takes it, 3 templates (a
    ragged template pair), a bad SFT in one of them, min_atoms 1 and 3: every cell of every
    template against the oracle, and against the same search with every window sum by the
    per-tau recurrence (tile code 1000)."""
    T = 3
    wl = tiny_workload(8000 + slots + grid.N_tau, slots, gaps, grid, n_templates=T, phi_random=True)
    atoms, t = wl.data.atoms.copy(), wl.data.t
    atoms[2, :, len(t) // 2] = np.nan  # template 2: one bad SFT (every channel, R19)
    grouped = pkg.plan_info(EXP, len(t), T, grid, exp_method=SCAN, tile=(0, 0, seg_len))
    plain = pkg.plan_info(EXP, len(t), T, grid, exp_method=SCAN, tile=(1000, 0, seg_len))
    assert grouped["n_launches"] == plain["n_launches"] + 1  # the grouped kernel does run
    a, td = dev(atoms), dev(t)
    for min_atoms in (2, 1, 3):
        res = pkg.tfstat_search(a, td, EXP, grid, exp_method=SCAN, want_maps=True, want_flags=True,
                                min_atoms=min_atoms, tile=(0, 0, seg_len))
        ref_k = pkg.tfstat_search(a, td, EXP, grid, exp_method=SCAN, want_maps=True, want_flags=True,
                                  min_atoms=min_atoms, tile=(1000, 0, seg_len))
        torch.cuda.synchronize()
        assert torch.equal(res.flags, ref_k.flags)
        assert not torch.equal(res.maps, ref_k.maps)  # another kernel summed the windows
        worst = 0.0
        for k in range(T):
            with np.errstate(invalid="ignore"):
                ref = oracle.map2F(atoms[k], t, EXP, grid, min_atoms=min_atoms)
            what = f"grouped window sums {grid} min_atoms {min_atoms} tpl{k}"
            worst = max(worst, check_cells(res.maps[k].cpu().numpy(), res.flags[k].cpu().numpy(),
                                           ref, what))
            check_result(res.numpy()[k], ref["twoF"], ref["flags"], grid.N_tau, what)
        assert worst < 0.25, worst  # (fraction of the tolerance used by the worst cell)


def test_exp_scan_work_counters(pkg):
    """tfstat_opts.stats (what bench.py's roofline of the sliding path is computed from): the
    kernels count what they executed.  Per-tau window sums: exactly the atoms of the last row's
    windows; cells: every cell once; grouped window sums: 8 moments x the atoms of each group's
    LONGEST window."""
    grid = Grid(0, 1800, 20, 1800, 1800, 700)
    T = 4
    wl = tiny_workload(8100, 2400, 0.1, grid, n_templates=T, phi_random=True)
    a, t = dev(wl.data.atoms), dev(wl.data.t)
    ref = oracle.map2F(wl.data.atoms[0], wl.data.t, EXP, grid)
    last = ref["cnt"][grid.N_t0 - 1].astype(np.int64)  # atoms per window of the last t0
    st = torch.zeros(pkg.binding.N_STATS, dtype=torch.int64, device="cuda")
    pkg.tfstat_search(a, t, EXP, grid, exp_method=SCAN, tile=(1000, 0, 0), stats=st)
    v = dict(zip(pkg.binding.STAT_NAMES, (int(x) for x in st.cpu().numpy())))
    assert v["terms_window"] == T * int(last.sum()) and v["terms_moment"] == 0
    assert v["cells"] == T * grid.n_cells
    # every step of every (template, tau) lets at most dt0 / T_SFT = 1 atom in and one out
    assert 0 < v["terms_enter"] <= T * grid.N_tau * (grid.N_t0 - 1)
    assert 0 < v["terms_leave"] <= T * grid.N_tau * (grid.N_t0 - 1)
    st.zero_()
    pkg.tfstat_search(a, t, EXP, grid, exp_method=SCAN, stats=st)
    w = dict(zip(pkg.binding.STAT_NAMES, (int(x) for x in st.cpu().numpy())))
    # tau >= 1.5 (R - 1) dtau / 0.17 in groups of R = 16, 32 and 64
    n16, n32, n64 = (int(np.ceil((1.5 * (R - 1) * grid.dtau / 0.17 - grid.tau_min) / grid.dtau))
                     for R in (16, 32, 64))
    assert (n16, n32, n64) == (132, 273, 555)
    assert w["terms_window"] == T * int(last[:n16].sum())
    groups = [(n, min(n + 16, n32)) for n in range(n16, n32, 16)] + \
             [(n, min(n + 32, n64)) for n in range(n32, n64, 32)] + \
             [(n, min(n + 64, grid.N_tau)) for n in range(n64, grid.N_tau, 64)]
    assert w["terms_moment"] == T * 8 * sum(int(last[b - 1]) for _, b in groups)
    assert (w["cells"], w["terms_enter"], w["terms_leave"]) == (v["cells"], v["terms_enter"],
                                                                 v["terms_leave"])


def test_exp_scan_config2_full(pkg):
    wl = make_workload(2)
    atoms, t = wl.data.atoms[0], wl.data.t
    ref = oracle.map2F(atoms, t, EXP, wl.grid)
    m, f = run_map(pkg, atoms, t, EXP, wl.grid, exp_method=SCAN)
    worst = check_cells(m, f, ref, "scan cfg2")
    assert worst < 0.5
    res = pkg.tfstat_search(dev(atoms[None]), dev(t), EXP, wl.grid, exp_method=SCAN)
    check_result(res.numpy()[0], ref["twoF"], ref["flags"], wl.grid.N_tau, "scan cfg2")


def test_exp_scan_config3_sampled(pkg):
    wl = make_workload(3)
    atoms, t = wl.data.atoms[0], wl.data.t
    m, f = run_map(pkg, atoms, t, EXP, wl.grid, exp_method=SCAN)
    ms, ns = _sample_cells(wl.grid, 30000, 3)
    ref = oracle.cells(atoms, t, EXP, wl.grid, ms, ns)
    worst = check_cells(m[ms, ns], f[ms, ns], ref, "scan cfg3 sampled")
    assert worst < 0.5
    full = oracle.map2F(atoms, t, EXP, wl.grid)  # the oracle's full map: a few seconds
    assert check_cells(m, f, full, "scan cfg3") < 0.5
    res = pkg.tfstat_search(dev(atoms[None]), dev(t), EXP, wl.grid, exp_method=SCAN).numpy()[0]
    check_result(res, full["twoF"], full["flags"], wl.grid.N_tau, "scan cfg3")


def test_exp_scan_config4_subset(pkg):
    from synth.configs import cfg4_injection_plan

    plan = cfg4_injection_plan()
    idx = sorted(set([0, 1, 2, 3] + sorted(plan)[:2]))
    wl = make_workload(4, templates=idx)
    res = pkg.tfstat_search(dev(wl.data.atoms), dev(wl.data.t), EXP, wl.grid,
                            exp_method=SCAN).numpy()
    for j, k in enumerate(idx):
        ref = oracle.map2F(wl.data.atoms[j], wl.data.t, EXP, wl.grid)
        check_result(res[j], ref["twoF"], ref["flags"], wl.grid.N_tau, f"scan cfg4 tpl{k}")


def test_exp_scan_config5_sampled(pkg):
    wl = make_workload(5)
    atoms, t = wl.data.atoms[0], wl.data.t
    res = pkg.tfstat_search(dev(atoms[None]), dev(t), EXP, wl.grid, exp_method=SCAN,
                            want_maps=True, want_flags=True)
    torch.cuda.synchronize()
    m, f = res.maps[0].cpu().numpy(), res.flags[0].cpu().numpy()
    ms, ns = _sample_cells(wl.grid, 20000, 55)
    ref = oracle.cells(atoms, t, EXP, wl.grid, ms, ns)
    worst = check_cells(m[ms, ns], f[ms, ns], ref, "scan cfg5 sampled")
    assert worst < 0.5
    _check_against_stored_oracle_marginals(res.numpy()[0], "cfg5_exp_marginals.txt", wl, EXP)
    _check_fused_equals_own_map(res.numpy()[0], m, f, wl.grid)
