"""Pins for the general-window / explicit-grid oracle (oracle_tfstat_map_general; SURVEY.md 8(f)
item 2; "variable sampling", "different window functions").

None re-uses the general oracle's code: its special cases must reproduce the already-pinned
rect / exp oracle exactly, and the table window is checked against an independent dense numpy
formulation built on numpy.interp.
"""
import numpy as np
import pytest

import oracle
from oracle.binding import TABLE, map2F_general
from synth import TSFT, Grid, tiny_workload

RECT, EXP = oracle.RECT, oracle.EXP


def _wl(seed=31, slots=90, gaps=0.15, grid=Grid(0, TSFT, 7, 2 * TSFT, TSFT, 9)):
    wl = tiny_workload(seed, slots, gaps, grid)
    return wl.data.atoms[0], wl.data.t, grid


@pytest.mark.parametrize("window,support", [(RECT, (1, 1)), (EXP, (3, 1))])
def test_uniform_arrays_reproduce_the_paper_windows_exactly(window, support):
    """(rect, 1 tau) and (exp, 3 tau) on arrays that spell out a uniform grid are eqs. (3), (4):
    same atoms, same order of summation => bit-identical to the pinned oracle."""
    atoms, t, g = _wl()
    ref = oracle.map2F(atoms, t, window, g)
    got = map2F_general(atoms, t, window, support, g.t0(), g.tau())
    for k in ("twoF", "flags", "cnt", "cond"):
        assert np.array_equal(got[k], ref[k]), k


def test_table_of_ones_is_the_rectangular_window():
    atoms, t, g = _wl(seed=32)
    ref = oracle.map2F(atoms, t, RECT, g)
    got = map2F_general(atoms, t, TABLE, (1, 1), g.t0(), g.tau(), table=np.ones(5, np.float32))
    assert np.array_equal(got["twoF"], ref["twoF"]) and np.array_equal(got["flags"], ref["flags"])


def test_fine_table_of_exp_tends_to_the_exponential_window():
    """Linear interpolation of exp(-u) on 3/4096 steps errs by <= h^2/8 = 6.7e-8 in the weight."""
    atoms, t, g = _wl(seed=33)
    ref = oracle.map2F(atoms, t, EXP, g)
    u = np.linspace(0.0, 3.0, 4097)
    got = map2F_general(atoms, t, TABLE, (3, 1), g.t0(), g.tau(),
                        table=np.exp(-u).astype(np.float32))
    assert np.array_equal(got["flags"], ref["flags"]) and np.array_equal(got["cnt"], ref["cnt"])
    ok = ref["flags"] == 0
    assert np.max(np.abs(got["twoF"] - ref["twoF"])[ok] / np.maximum(1.0, ref["twoF"][ok])) < 1e-5


def _dense_table(atoms, t, sup, table, t0g, taug, min_atoms=2):
    """Independent formulation: dense [cells x atoms] weights via numpy.interp, sums by einsum,
    2F = 2 v^H M^-1 v by a 2x2 solve (eq. 6)."""
    a = atoms.astype(np.float64)
    tt = t.astype(np.int64)[None, None, :]
    t0 = np.asarray(t0g, np.int64)[:, None, None]
    tau = np.asarray(taug, np.int64)[None, :, None]
    dt = tt - t0
    inside = (dt >= 0) & (dt * sup[1] < sup[0] * tau)
    knots = np.linspace(0.0, sup[0] / sup[1], len(table))
    W = np.where(inside, np.interp(np.where(inside, dt, 0) / tau.astype(np.float64), knots,
                                   np.asarray(table, np.float64)), 0.0)
    ABC = np.einsum("mna,ca->mnc", W * W, a[0:3])
    Fa = np.einsum("mna,a->mn", W, a[3] + 1j * a[4])
    Fb = np.einsum("mna,a->mn", W, a[5] + 1j * a[6])
    cnt = inside.sum(-1)
    twoF = np.zeros(cnt.shape)
    flags = np.zeros(cnt.shape, np.uint8)
    for m in range(cnt.shape[0]):
        for n in range(cnt.shape[1]):
            A, B, Cc = ABC[m, n]
            M = np.array([[A, Cc], [Cc, B]])
            flags[m, n] = (cnt[m, n] < min_atoms) | (2 * (not (A * B - Cc * Cc > 0)))
            if flags[m, n] == 0:
                v = np.array([Fa[m, n], Fb[m, n]])
                twoF[m, n] = 2.0 * np.real(np.conj(v) @ np.linalg.solve(M, v))
    return twoF, flags, cnt


@pytest.mark.parametrize("sup", [(5, 2), (1, 1), (7, 3)])
def test_table_window_on_irregular_grids_against_dense_numpy(sup):
    """A power-law-like window (1+u)^-1.5 sampled coarsely (so that interpolation matters), a
    rational support, unsorted / repeated / off-lattice t0 and tau values."""
    atoms, t, _ = _wl(seed=34, slots=120, gaps=0.2)
    rng = np.random.default_rng(5)
    t0g = np.array([0, 900, 5 * TSFT, 3 * TSFT + 17, 5 * TSFT, 40 * TSFT, -TSFT], np.int32)
    taug = np.sort(rng.integers(TSFT, 30 * TSFT, size=8)).astype(np.int32)[::-1].copy()
    table = ((1.0 + np.linspace(0.0, sup[0] / sup[1], 9)) ** -1.5).astype(np.float32)
    got = map2F_general(atoms, t, TABLE, sup, t0g, taug, table=table)
    twoF, flags, cnt = _dense_table(atoms, t, sup, table, t0g, taug)
    assert np.array_equal(got["cnt"], cnt)
    assert np.array_equal(got["flags"], flags)
    ok = flags == 0
    assert np.allclose(got["twoF"][ok], twoF[ok], rtol=1e-9, atol=1e-9)
    assert np.all(got["twoF"][~ok] == 0.0)
    # rows with the same t0 (indices 2 and 4) are identical: cells depend on (t0, tau) only
    assert np.array_equal(got["twoF"][2], got["twoF"][4])


def test_irregular_grid_cells_equal_the_uniform_grid_cells():
    """Any (t0, tau) pair taken from a uniform grid gives the uniform map's cell, whatever the
    order of the arrays (each cell depends on its own t0 and tau only)."""
    atoms, t, g = _wl(seed=35)
    ref = oracle.map2F(atoms, t, EXP, g)
    pm = np.array([4, 0, 6, 2]); pn = np.array([8, 3, 3, 0, 5])
    got = map2F_general(atoms, t, EXP, (3, 1), g.t0()[pm], g.tau()[pn])
    assert np.array_equal(got["twoF"], ref["twoF"][np.ix_(pm, pn)])
    assert np.array_equal(got["flags"], ref["flags"][np.ix_(pm, pn)])


def test_general_oracle_rejects_bad_arguments():
    atoms, t, g = _wl()
    with pytest.raises(ValueError):
        map2F_general(atoms, t, TABLE, (1, 1), g.t0(), g.tau())            # no table
    with pytest.raises(ValueError):
        map2F_general(atoms, t, EXP, (0, 1), g.t0(), g.tau())              # empty support
    with pytest.raises(ValueError):
        map2F_general(atoms, t, EXP, (3, 1), g.t0(), np.array([0, 1800]))  # tau < 1


# ----------------------------------------------------------------------------------------
# per-detector merge (oracle_merge_detectors)
# ----------------------------------------------------------------------------------------
def _detector_sets(seed=41, n_slots=300):
    from synth import make_detector_atoms

    rng = np.random.default_rng(seed)
    t = (np.arange(n_slots) * TSFT).astype(np.int32)
    per_det = make_detector_atoms(t, np.random.default_rng(seed + 1)).astype(np.float32)
    keep = [rng.random(n_slots) > 0.25, rng.random(n_slots) > 0.4]  # each detector's own gaps
    keep[0][:3] = False                                              # a slot neither detector has
    keep[1][:3] = False
    atoms = [np.ascontiguousarray(per_det[d][:, keep[d]]) for d in (0, 1)]
    ts = [t[keep[d]] for d in (0, 1)]
    return t, per_det, keep, atoms, ts


def test_merge_detectors_against_numpy_bit_exact():
    from oracle.binding import merge_detectors

    t, per_det, keep, atoms, ts = _detector_sets()
    t_out = np.union1d(ts[0], ts[1]).astype(np.int32)
    got = merge_detectors(atoms, ts, t_out)
    ref = np.zeros((7, len(t_out)), np.float32)
    for d in (0, 1):  # independent formulation: scatter by searchsorted, fp32 adds, same order
        ref[:, np.searchsorted(t_out, ts[d])] += atoms[d]
    assert got.dtype == np.float32 and np.array_equal(got, ref)
    # a time stamp nobody has gives zeros; atoms outside t_out are dropped
    t_odd = np.concatenate([[0], t_out[::2]]).astype(np.int32)
    got2 = merge_detectors(atoms, ts, t_odd)
    assert np.all(got2[:, 0] == 0.0) and np.array_equal(got2[:, 1:], ref[:, ::2])


def test_merged_detectors_reproduce_the_merged_atom_model():
    """Without gaps the merge of the per-detector atoms is synth.make_atoms (the model the five
    configs use), and the map of the merged set is the map of make_atoms within fp32 rounding."""
    from oracle.binding import merge_detectors
    from synth import make_atoms, make_detector_atoms

    t = (np.arange(200) * TSFT).astype(np.int32)
    per_det = make_detector_atoms(t, np.random.default_rng(7)).astype(np.float32)
    merged = merge_detectors([per_det[0], per_det[1]], [t, t], t)
    ref = make_atoms(t, np.random.default_rng(7)).astype(np.float32)
    assert np.allclose(merged, ref, rtol=3e-7, atol=3e-7)
    g = Grid(0, TSFT, 6, 4 * TSFT, 2 * TSFT, 7)
    a = oracle.map2F(merged, t, EXP, g)["twoF"]
    b = oracle.map2F(ref, t, EXP, g)["twoF"]
    assert np.allclose(a, b, rtol=1e-4, atol=1e-4)
