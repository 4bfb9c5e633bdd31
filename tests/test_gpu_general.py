"""GPU parity for tfstat_map_general (general windows on explicit grids) against the fp64 oracle
oracle_tfstat_map_general, element by element through the C ABI (-m gpu)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from oracle.binding import map2F_general  # noqa: E402
from synth import TSFT, Grid, make_workload, tiny_workload  # noqa: E402
from tests.parity import check_cells, check_result  # noqa: E402

pytestmark = pytest.mark.gpu

RECT, EXP, TABLE = 0, 1, 2


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


def power_law(sup, n):
    return ((1.0 + np.linspace(0.0, sup[0] / sup[1], n)) ** -1.5).astype(np.float32)


def run(pkg, atoms, t, kind, sup, t0g, taug, table=None, **kw):
    m, f, r = pkg.tfstat_map_general(dev(atoms), dev(t), kind, sup, dev(t0g), dev(taug),
                                     table=None if table is None else dev(table),
                                     want_flags=True, **kw)
    torch.cuda.synchronize()
    return m.cpu().numpy(), f.cpu().numpy(), r.numpy()[0]


CASES = [
    # kind, support, table samples (None: no table)
    (RECT, (1, 1), None),
    (EXP, (3, 1), None),
    (EXP, (5, 2), None),
    (TABLE, (5, 2), 9),        # coarse table: the interpolation matters
    (TABLE, (2, 1), 5000),     # table too large for shared memory: read through L1
]


@pytest.mark.parametrize("ct", [0, 1, 2, 4])
@pytest.mark.parametrize("kind,sup,ntab", CASES)
def test_general_irregular_grids(pkg, kind, sup, ntab, ct):
    """Unsorted, repeated, off-lattice t0 values (some before the data), 300 irregular tau values
    (three CTAs along tau with a ragged tail, long windows spanning several staged chunks)."""
    wl = tiny_workload(301, 1500, 0.2, Grid(0, TSFT, 1, TSFT, TSFT, 1))
    atoms, t = wl.data.atoms[0], wl.data.t
    rng = np.random.default_rng(7)
    t0g = np.concatenate([[0, -3 * TSFT, 900, 5 * TSFT, 5 * TSFT, 1400 * TSFT, 1600 * TSFT],
                          rng.integers(0, 1500 * TSFT, size=14)]).astype(np.int32)
    taug = rng.permutation(np.concatenate([[1, 1799, 1800, 1801],
                                           rng.integers(TSFT, 900 * TSFT, size=296)])).astype(np.int32)
    table = None if ntab is None else power_law(sup, ntab)
    m, f, r = run(pkg, atoms, t, kind, sup, t0g, taug, table, cells_per_thread=ct)
    ref = map2F_general(atoms, t, kind, sup, t0g, taug, table=table)
    check_cells(m, f, ref, f"general kind {kind}")
    check_result(r, ref["twoF"], ref["flags"], len(taug), f"general kind {kind}")


@pytest.mark.parametrize("window,sup", [(RECT, (1, 1)), (EXP, (3, 1))])
def test_general_equals_the_lattice_kernels_on_a_uniform_grid(pkg, window, sup):
    """The paper's two windows through the general entry point agree with tfstat_map (the
    lattice kernels) within the parity tolerance, and with the oracle."""
    grid = Grid(0, 1800, 23, 3600, 3600, 140)
    wl = tiny_workload(302, 600, 0.1, grid)
    atoms, t = wl.data.atoms[0], wl.data.t
    m, f, r = run(pkg, atoms, t, window, sup, grid.t0().astype(np.int32),
                  grid.tau().astype(np.int32))
    ref = oracle.map2F(atoms, t, window, grid)
    check_cells(m, f, ref, "general on uniform grid")
    m2, f2 = pkg.tfstat_map(dev(atoms), dev(t), window, grid, want_flags=True)
    assert np.array_equal(f, f2.cpu().numpy())
    np.testing.assert_allclose(m, m2.cpu().numpy(), rtol=2e-3, atol=2e-3)


def test_general_config2_sampled_rows(pkg):
    """BASELINE.json config 2 (1440 atoms, tau up to 20 days) on 6 of its t0 rows and all 937 tau."""
    wl = make_workload(2)
    atoms, t, g = wl.data.atoms[0], wl.data.t, wl.grid
    rows = np.array([0, 1, 191, 192, 300, 479])
    t0g = g.t0()[rows].astype(np.int32)
    taug = g.tau().astype(np.int32)
    m, f, r = run(pkg, atoms, t, EXP, (3, 1), t0g, taug)
    ref = oracle.map2F(atoms, t, EXP, g)
    sub = {k: v[rows] for k, v in ref.items()}
    check_cells(m, f, sub, "config 2 rows")
    check_result(r, sub["twoF"], sub["flags"], g.N_tau, "config 2 rows")


def test_general_degenerate_and_errors(pkg):
    wl = tiny_workload(303, 40, 0.0, Grid(0, TSFT, 1, TSFT, TSFT, 1))
    atoms, t = wl.data.atoms[0], wl.data.t
    # windows after the data, a non-positive tau, a one-atom window: flagged, never an error
    t0g = np.array([100 * TSFT, 0, 0], np.int32)
    taug = np.array([TSFT, 0, -5, 1800, 3600], np.int32)
    m, f, r = run(pkg, atoms, t, EXP, (1, 1), t0g, taug)
    assert np.all(f[0] == 3) and np.all(m[0] == 0.0)          # empty windows
    assert np.all(f[1:, :3] != 0) and np.all(m[1:, :3] == 0.0)  # tau < 1, and tau = 1 (1 atom)
    assert f[1, 3] == 1 and f[1, 4] == 0                        # 1 atom / 2 atoms
    assert r["n_valid"] == int((f == 0).sum())
    # marginals only, map only
    m2, f2, r2 = pkg.tfstat_map_general(dev(atoms), dev(t), EXP, (1, 1), dev(t0g), dev(taug),
                                        want_map=False)
    assert m2 is None and np.array_equal(r2.numpy(), np.array([r]))
    with pytest.raises(pkg.TfstatError):
        pkg.tfstat_map_general(dev(atoms), dev(t), TABLE, (1, 1), dev(t0g), dev(taug))  # no table
    with pytest.raises(pkg.TfstatError):
        pkg.tfstat_map_general(dev(atoms), dev(t), EXP, (0, 1), dev(t0g), dev(taug))
    with pytest.raises(pkg.TfstatError):
        pkg.tfstat_map_general(dev(atoms), dev(t), 7, (1, 1), dev(t0g), dev(taug))


def test_merge_detectors_bit_exact_and_end_to_end(pkg):
    """tfstat_merge_detectors against oracle_merge_detectors, bit for bit (fp32 adds in a fixed
    order), batched over templates with detectors that have their own gaps; then the merged atoms
    through tfstat_search against the oracle's map of the oracle's merge."""
    from oracle.binding import merge_detectors
    from synth import make_detector_atoms

    n_slots, T = 700, 3
    t = (np.arange(n_slots) * TSFT).astype(np.int32)
    rng = np.random.default_rng(11)
    keep = [rng.random(n_slots) > 0.2, rng.random(n_slots) > 0.35, rng.random(n_slots) > 0.5]
    for k in keep:
        k[100:130] = False  # a common gap: time stamps nobody has do not appear in the union
    per = [np.stack([make_detector_atoms(t, np.random.default_rng(100 + 10 * tpl), phi=0.3 * tpl)
                     .astype(np.float32) for tpl in range(T)]) for _ in range(1)][0]  # [T, 2, 7, N]
    # three "detectors": the model's two, and a second copy of detector 0 scaled (a third site)
    dets = [per[:, 0][:, :, keep[0]], per[:, 1][:, :, keep[1]], 0.5 * per[:, 0][:, :, keep[2]]]
    ts = [t[k] for k in keep]
    t_out = np.union1d(np.union1d(ts[0], ts[1]), ts[2]).astype(np.int32)
    assert len(t_out) < n_slots
    got = pkg.tfstat_merge_detectors([dev(d) for d in dets], [dev(x) for x in ts], dev(t_out))
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    for tpl in range(T):
        ref = merge_detectors([d[tpl] for d in dets], ts, t_out)
        assert np.array_equal(got[tpl], ref), f"template {tpl}: merge differs from the oracle"
    # single-template form, and a t_out with a stamp nobody has / without some stamps
    t_odd = np.concatenate([[-TSFT], t_out[::3]]).astype(np.int32)
    g1 = pkg.tfstat_merge_detectors([dev(d[0]) for d in dets], [dev(x) for x in ts], dev(t_odd))
    assert np.array_equal(g1.cpu().numpy(), merge_detectors([d[0] for d in dets], ts, t_odd))
    # end to end: merged atoms -> search
    grid = Grid(0, TSFT, 30, 4 * TSFT, 2 * TSFT, 150)
    res = pkg.tfstat_search(dev(got), dev(t_out), EXP, grid, want_maps=True, want_flags=True)
    for tpl in range(T):
        ref = oracle.map2F(got[tpl], t_out, EXP, grid)
        check_cells(res.maps[tpl].cpu().numpy(), res.flags[tpl].cpu().numpy(), ref, f"merged {tpl}")
    with pytest.raises(pkg.TfstatError):
        pkg.tfstat_merge_detectors([dev(dets[0])] * 9, [dev(ts[0])] * 9, dev(t_out))  # > 8 detectors
