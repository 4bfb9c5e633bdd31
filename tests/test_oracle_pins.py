"""Pins for the fp64 oracle: things the paper and the mathematics fix, none of which
re-use the oracle's own formula or code.

Each test is chosen so that a plausible mistake in oracle/tfstat_oracle.c (dropped term,
wrong sign/index, w vs w^2, closed vs half-open window, transposed map) fails it.
"""
from fractions import Fraction

import numpy as np
import pytest
from scipy import stats
from scipy.special import logsumexp

import oracle
from synth import (TSFT, Grid, antenna_terms, inject_exponential, inject_rectangular,
                   make_atoms, make_workload, tiny_workload)
from tests.golden.load_golden import load

RECT, EXP = oracle.RECT, oracle.EXP


# ----------------------------------------------------------------------------------------
# independent formulations used as pins
# ----------------------------------------------------------------------------------------
def dense_bruteforce(atoms, t, window, grid, min_atoms=2):
    """I8: dense [cells x atoms] weight matrix times the atom matrix, then a 2x2 complex
    linear solve per cell: 2F = 2 v^H M^{-1} v with M=[[A,C],[C,B]], v=(Fa,Fb) -- eq. (6),
    PAPER.md:61, specialised as in eq. (7).  No loops over atoms, no explicit eq. (7)."""
    a = atoms.astype(np.float64)
    t = t.astype(np.int64)
    k = 3 if window == EXP else 1
    t0 = grid.t0()[:, None, None]
    tau = grid.tau()[None, :, None]
    tt = t[None, None, :]
    inside = (tt >= t0) & (tt < t0 + k * tau)
    if window == EXP:
        W = np.where(inside, np.exp(-np.where(inside, tt - t0, 0) / tau.astype(np.float64)), 0.0)
    else:
        W = inside.astype(np.float64)
    ABC = np.einsum("mna,ca->mnc", W * W, a[0:3])
    Fa = np.einsum("mna,a->mn", W, a[3] + 1j * a[4])
    Fb = np.einsum("mna,a->mn", W, a[5] + 1j * a[6])
    cnt = inside.sum(-1)
    twoF = np.zeros((grid.N_t0, grid.N_tau))
    flags = np.zeros((grid.N_t0, grid.N_tau), np.uint8)
    for m in range(grid.N_t0):
        for n in range(grid.N_tau):
            A, B, Cc = ABC[m, n]
            M = np.array([[A, Cc], [Cc, B]])
            if cnt[m, n] < min_atoms:
                flags[m, n] |= 1
            if not (np.linalg.det(M) > 0):
                flags[m, n] |= 2
            if flags[m, n]:
                continue
            v = np.array([Fa[m, n], Fb[m, n]])
            twoF[m, n] = 2.0 * np.real(np.conj(v) @ np.linalg.solve(M, v))
    return twoF, flags, cnt


def exact_rect_cell(atoms_frac, t, t0, tau):
    """Exact rational rect cell: plain sums of the atoms in [t0, t0+tau), then eq. (7)."""
    idx = [i for i, ti in enumerate(t) if t0 <= ti < t0 + tau]
    S = [sum((atoms_frac[r][i] for i in idx), Fraction(0)) for r in range(7)]
    A, B, Cc, far, fai, fbr, fbi = S
    D = A * B - Cc * Cc
    if len(idx) < 2 or D <= 0:
        return None, len(idx)
    F = (B * (far * far + fai * fai) + A * (fbr * fbr + fbi * fbi)
         - 2 * Cc * (far * fbr + fai * fbi)) / D
    return 2 * F, len(idx)


def toy_inputs():
    g = load("T0_toy.txt")
    atoms = np.stack([g[k] for k in ("a2", "b2", "ab", "FaRe", "FaIm", "FbRe", "FbIm")])
    atoms32 = atoms.astype(np.float32)
    assert np.array_equal(atoms32.astype(np.float64), atoms)  # exactly representable
    t = g["t_atoms"].astype(np.int32)
    t0_min, dt0, N_t0 = (int(x) for x in g["grid_t0"])
    tau_min, dtau, N_tau = (int(x) for x in g["grid_tau"])
    return g, atoms32, t, Grid(t0_min, dt0, N_t0, tau_min, dtau, N_tau)


# ----------------------------------------------------------------------------------------
# T0 golden + exact rational arithmetic
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("wname,window", [("rect", RECT), ("exp", EXP)])
def test_T0_golden(wname, window):
    g, atoms, t, grid = toy_inputs()
    r = oracle.map2F(atoms, t, window, grid)
    assert np.array_equal(r["cnt"].ravel(), g[f"{wname}_cnt"].astype(int))
    assert np.array_equal((r["flags"].ravel() != 0).astype(int), g[f"{wname}_flagged"].astype(int))
    np.testing.assert_allclose(r["twoF"].ravel(), g[f"{wname}_2F"], rtol=0, atol=2e-12)
    mg = oracle.marginalise(r["twoF"], r["flags"])
    assert mg.m * grid.N_tau + mg.n == int(g[f"{wname}_argmax_flat"][0])
    assert mg.n_valid == int(g[f"{wname}_n_valid"][0])
    assert abs(mg.max2F - g[f"{wname}_max2F"][0]) < 1e-9
    assert abs(mg.logB - g[f"{wname}_logB"][0]) < 2e-12


def test_T0_rect_exact_rational():
    g, atoms, t, grid = toy_inputs()
    fr = [[Fraction(float(x)) for x in row] for row in atoms]
    r = oracle.map2F(atoms, t, RECT, grid)
    for m in range(grid.N_t0):
        for n in range(grid.N_tau):
            ex, cnt = exact_rect_cell(fr, [int(x) for x in t], int(grid.t0()[m]), int(grid.tau()[n]))
            assert cnt == r["cnt"][m, n]
            if ex is None:
                assert r["flags"][m, n] != 0 and r["twoF"][m, n] == 0.0
            else:
                assert r["flags"][m, n] == 0
                assert abs(r["twoF"][m, n] - float(ex)) <= 4e-15 * max(1.0, float(ex))
    assert exact_rect_cell(fr, [int(x) for x in t], 0, 3600)[0] == Fraction(620, 99)


def test_rect_exact_rational_random():
    """Random dyadic atoms (exact in fp32 and in Fraction), gaps, non-unit grid steps."""
    rng = np.random.default_rng(7)
    slots = np.sort(rng.choice(40, size=26, replace=False))
    t = (slots * 1800).astype(np.int32)
    a = rng.integers(1, 64, size=(2, t.size)) / 64.0
    b = rng.integers(-64, 64, size=(2, t.size)) / 64.0
    nre = rng.integers(-128, 128, size=(2, t.size)) / 32.0
    nim = rng.integers(-128, 128, size=(2, t.size)) / 32.0
    nd = nre + 1j * nim
    atoms = np.stack([(a * a).sum(0), (b * b).sum(0), (a * b).sum(0), (a * nd).sum(0).real,
                      (a * nd).sum(0).imag, (b * nd).sum(0).real, (b * nd).sum(0).imag])
    atoms32 = atoms.astype(np.float32)
    assert np.array_equal(atoms32.astype(np.float64), atoms)
    grid = Grid(-1800, 2700, 9, 1800, 4500, 7)
    fr = [[Fraction(float(x)) for x in row] for row in atoms32]
    r = oracle.map2F(atoms32, t, RECT, grid)
    n_checked = 0
    for m in range(grid.N_t0):
        for n in range(grid.N_tau):
            ex, cnt = exact_rect_cell(fr, [int(x) for x in t], int(grid.t0()[m]), int(grid.tau()[n]))
            assert cnt == r["cnt"][m, n]
            if ex is not None:
                n_checked += 1
                assert abs(r["twoF"][m, n] - float(ex)) <= 1e-12 * max(1.0, float(ex))
            else:
                assert r["flags"][m, n] != 0
    assert n_checked > 40


# ----------------------------------------------------------------------------------------
# I8 brute force by an independent formulation, tiny grids, gaps, ragged edges
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("window", [RECT, EXP])
@pytest.mark.parametrize("seed,gaps,grid", [
    (11, 0.0, Grid(0, 1800, 12, 3600, 1800, 10)),
    (12, 0.3, Grid(-5400, 2700, 17, 1800, 3100, 13)),     # off-lattice steps, starts before data
    (13, 0.2, Grid(30 * 1800, 900, 40, 2 * 1800, 7200, 6)),  # windows overrun the data end
])
def test_bruteforce_dense(window, seed, gaps, grid):
    wl = tiny_workload(seed, 64, gaps, grid)
    atoms, t = wl.data.atoms[0], wl.data.t
    twoF, flags, cnt = dense_bruteforce(atoms, t, window, grid)
    r = oracle.map2F(atoms, t, window, grid)
    assert np.array_equal(r["cnt"], cnt)
    assert np.array_equal(r["flags"], flags)
    np.testing.assert_allclose(r["twoF"], twoF, rtol=1e-10, atol=1e-10)
    # the cell-list entry point is the same function
    ms, ns = np.meshgrid(np.arange(grid.N_t0), np.arange(grid.N_tau), indexing="ij")
    rc = oracle.cells(atoms, t, window, grid, ms.ravel(), ns.ravel())
    assert np.array_equal(rc["twoF"], r["twoF"].ravel())
    assert np.array_equal(rc["flags"], r["flags"].ravel())


# ----------------------------------------------------------------------------------------
# I1 closed form for injections, I1b peak recovery
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("window,inject", [(EXP, inject_exponential), (RECT, inject_rectangular)])
def test_injection_closed_form(window, inject):
    """Noise-free atoms Fa = W(c1 a2 + c2 ab), Fb = W(c1 ab + c2 b2): at the matched cell
    2F = rho^2 exactly, everywhere else 2F <= rho^2 (Cauchy-Schwarz); argmax = injected cell."""
    t = (np.arange(200) * TSFT).astype(np.int32)
    rng = np.random.default_rng(5)
    atoms = make_atoms(t, rng, noise=False).astype(np.float32)
    grid = Grid(0, 1800, 30, 7200, 3600, 20)
    m_inj, n_inj, rho = 11, 7, 10.0
    inject(atoms, t, int(grid.t0()[m_inj]), int(grid.tau()[n_inj]), rho, rng)
    r = oracle.map2F(atoms, t, window, grid)
    # fp32 rounding of the injected Fa, Fb limits the match to ~1e-6 relative
    assert abs(r["twoF"][m_inj, n_inj] - rho ** 2) < 2e-5 * rho ** 2
    assert r["twoF"].max() <= rho ** 2 * (1 + 2e-5)
    mg = oracle.marginalise(r["twoF"], r["flags"])
    assert (mg.m, mg.n) == (m_inj, n_inj)


def test_config2_peak_recovery_with_noise():
    """I1b on BASELINE.json configs[1]: injected (t0,tau)=(4 d, 6 d) is cell (192, 264); with
    noise the peak is >= the injected cell's 2F, close in t0; E[2F]=4+rho^2 at that cell."""
    wl = make_workload(2)
    (m_inj, n_inj, rho), = wl.injections.values()
    assert (m_inj, n_inj) == (192, 264)
    atoms, t = wl.data.atoms[0], wl.data.t
    ms = np.repeat(np.arange(m_inj - 24, m_inj + 25), 9)
    ns = np.tile(np.arange(n_inj - 200, n_inj + 201, 50), 49)
    r = oracle.cells(atoms, t, EXP, wl.grid, ms, ns)
    k = int(np.argmax(r["twoF"]))
    at_inj = r["twoF"][(ms == m_inj) & (ns == n_inj)][0]
    assert r["twoF"][k] >= at_inj
    assert abs(int(ms[k]) - m_inj) <= 6
    # non-central chi^2_4 with rho^2 = 100: sd = sqrt(2(4+2*100)) ~ 20
    assert abs(at_inj - (4 + rho ** 2)) < 5 * np.sqrt(2 * (4 + 2 * rho ** 2))


# ----------------------------------------------------------------------------------------
# I2 full-span rectangular window == CW F-statistic from total sums
# ----------------------------------------------------------------------------------------
def test_full_span_rect_is_cw_fstat():
    wl = make_workload(1)
    atoms, t = wl.data.atoms[0].astype(np.float64), wl.data.t
    S = atoms.sum(1)
    A, B, Cc = S[0], S[1], S[2]
    Fa, Fb = complex(S[3], S[4]), complex(S[5], S[6])
    M = np.array([[A, Cc], [Cc, B]])
    v = np.array([Fa, Fb])
    cw = 2.0 * np.real(np.conj(v) @ np.linalg.inv(M) @ v)
    full = oracle.map2F(wl.data.atoms[0], t, RECT, Grid(0, 1800, 1, 48 * TSFT, 1, 1))
    assert full["cnt"][0, 0] == 48  # t0 = 0, tau = 24 h: the whole data set
    assert abs(full["twoF"][0, 0] - cw) < 1e-12 * cw
    r = oracle.map2F(wl.data.atoms[0], t, RECT, wl.grid)
    assert r["cnt"][0, -1] == 24 and r["cnt"][23, -1] == 24 and r["cnt"][23, 0] == 1
    # config 1's tau = T_SFT column holds 1 atom per cell and is flagged
    assert np.all(r["flags"][:, 0] == 1) and np.all(r["twoF"][:, 0] == 0.0)
    assert np.count_nonzero(r["flags"]) == 24


# ----------------------------------------------------------------------------------------
# I4 / I5 invariances
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("window", [RECT, EXP])
def test_time_shift_and_amplitude_scaling(window):
    grid = Grid(1800, 1800, 10, 3600, 1800, 9)
    wl = tiny_workload(21, 48, 0.15, grid)
    atoms, t = wl.data.atoms[0], wl.data.t
    base = oracle.map2F(atoms, t, window, grid)
    # I4: shift every time by the same offset
    sh = 123456
    g2 = Grid(grid.t0_min + sh, grid.dt0, grid.N_t0, grid.tau_min, grid.dtau, grid.N_tau)
    r2 = oracle.map2F(atoms, (t + sh).astype(np.int32), window, g2)
    assert np.array_equal(r2["twoF"], base["twoF"]) and np.array_equal(r2["cnt"], base["cnt"])
    # I5: (a2,b2,ab) x s^2 and (Fa,Fb) x s leave F unchanged (s = 4: exact in fp32)
    a3 = atoms.copy()
    a3[0:3] *= 16.0
    a3[3:7] *= 4.0
    r3 = oracle.map2F(a3, t, window, grid)
    np.testing.assert_allclose(r3["twoF"], base["twoF"], rtol=1e-12)
    # (Fa,Fb) x s alone scales F by s^2
    a4 = atoms.copy()
    a4[3:7] *= 4.0
    r4 = oracle.map2F(a4, t, window, grid)
    np.testing.assert_allclose(r4["twoF"], 16.0 * base["twoF"], rtol=1e-12)
    # swapping the roles (a<->b, Fa<->Fb) is a symmetry of eq. (7)
    a5 = atoms[[1, 0, 2, 5, 6, 3, 4]]
    r5 = oracle.map2F(a5, t, window, grid)
    np.testing.assert_allclose(r5["twoF"], base["twoF"], rtol=1e-12)


# ----------------------------------------------------------------------------------------
# I6 integer term counts equal eqs. (A.5)/(A.6) on gapless data
# ----------------------------------------------------------------------------------------
def _A6(grid, T_data, k):
    t0 = grid.t0()[:, None]
    tau = grid.tau()[None, :]
    return int((np.minimum(T_data - t0, k * tau) // TSFT).sum())


def test_term_counts_A6_config2_and_config4():
    """PAPER.md:240 eq. (A.6); SURVEY.md quotes 436 248 960 (config 2) and 263 240 064 per
    template (config 4) for half-open windows."""
    wl = make_workload(2)
    r = oracle.map2F(wl.data.atoms[0], wl.data.t, EXP, wl.grid)
    assert int(r["cnt"].sum()) == _A6(wl.grid, 1440 * TSFT, 3) == 436248960
    # embedded-case reduction 3 N_t0 N_tau (tau_min + 0.5 Delta tau)/T_SFT
    g = wl.grid
    assert g.t0()[-1] + 3 * g.tau()[-1] > 1440 * TSFT  # config 2 is NOT embedded
    wl4 = make_workload(4, templates=[0])
    ms, ns = np.meshgrid(np.arange(96), np.arange(1417), indexing="ij")
    r4 = oracle.cells(wl4.data.atoms[0], wl4.data.t, EXP, wl4.grid, ms.ravel(), ns.ravel())
    assert int(r4["cnt"].sum()) == _A6(wl4.grid, 2880 * TSFT, 3) == 263240064


def test_term_counts_A5_rect_and_embedded_case():
    """PAPER.md:234 eq. (A.5) counts the paper's running-sum steps: per t0 the atoms of the
    longest window.  Embedded case: N_t0 tau_max / T_SFT."""
    t = (np.arange(100) * TSFT).astype(np.int32)
    atoms = make_atoms(t, np.random.default_rng(1)).astype(np.float32)
    grid = Grid(0, 1800, 20, 3600, 1800, 30)  # t0_max + tau_max = 19+31 = 50 slots < 100
    r = oracle.map2F(atoms, t, RECT, grid)
    assert int(r["cnt"][:, -1].sum()) == grid.N_t0 * int(grid.tau()[-1]) // TSFT
    assert np.array_equal(r["cnt"], np.broadcast_to(grid.tau()[None, :] // TSFT, r["cnt"].shape))
    grid2 = Grid(0, 1800, 98, 3600, 1800, 98)  # the paper's timing setup
    r2 = oracle.map2F(atoms, t, RECT, grid2)
    A5 = int((np.minimum(100 * TSFT - grid2.t0(), grid2.tau()[-1]) // TSFT).sum())
    assert int(r2["cnt"][:, -1].sum()) == A5
    r3 = oracle.map2F(atoms, t, EXP, grid)  # exp: 3 tau / T_SFT atoms per cell
    assert np.array_equal(r3["cnt"], np.minimum(3 * grid.tau()[None, :] // TSFT,
                                                100 - grid.t0()[:, None] // TSFT))


# ----------------------------------------------------------------------------------------
# conventions: half-open edges, truncation, degenerate cells
# ----------------------------------------------------------------------------------------
def test_half_open_edges_and_empty_windows():
    t = np.array([0, 1800, 3600, 9000], dtype=np.int32)
    atoms = make_atoms(t, np.random.default_rng(3)).astype(np.float32)
    # [0,3600): atom at 3600 excluded; [0,3601): included; [1,3601), [1,3602): atom at 0
    # excluded, atom at 3600 included
    r = oracle.map2F(atoms, t, RECT, Grid(0, 1, 2, 3600, 1, 2))
    assert r["cnt"].tolist() == [[2, 3], [2, 2]]
    # exp window of tau covers [t0, t0 + 3 tau)
    r = oracle.map2F(atoms, t, EXP, Grid(0, 1, 1, 1200, 1, 2))
    assert r["cnt"].tolist() == [[2, 3]]
    # before the data, in a gap, after the data: empty, flagged, 2F = 0, no error
    r = oracle.map2F(atoms, t, RECT, Grid(-100000, 104000, 3, 1800, 1, 1))
    assert r["cnt"].ravel().tolist() == [0, 0, 0]
    assert np.all(r["flags"] == 3) and np.all(r["twoF"] == 0)
    mg = oracle.marginalise(r["twoF"], r["flags"])
    assert (mg.n_valid, mg.m, mg.n, mg.max2F) == (0, -1, -1, 0.0) and mg.logB == -np.inf


def test_single_detector_degenerate_and_exactly_determined():
    """One single-detector atom: D = a^2 b^2 - (ab)^2 = 0 exactly (flag bit 1 even with
    min_atoms = 1).  I7: two single-detector atoms determine the 4 amplitudes exactly, so
    F = sum |n|^2 whatever the weights (rect and exp agree)."""
    t = np.array([0, 1800], dtype=np.int32)
    a = np.array([0.5, 0.75])
    b = np.array([0.25, -0.5])
    n = np.array([0.5 - 1.25j, -0.75 + 0.5j])
    atoms = np.stack([a * a, b * b, a * b, (a * n).real, (a * n).imag, (b * n).real,
                      (b * n).imag]).astype(np.float32)
    g1 = Grid(0, 1800, 1, 1800, 1800, 1)
    r = oracle.map2F(atoms, t, RECT, g1, min_atoms=1)
    assert r["cnt"][0, 0] == 1 and r["flags"][0, 0] == 2 and r["twoF"][0, 0] == 0
    expect = 2.0 * float((abs(n) ** 2).sum())
    for window, g in ((RECT, Grid(0, 1800, 1, 3600, 1800, 1)), (EXP, Grid(0, 1800, 1, 1800, 700, 3))):
        r = oracle.map2F(atoms, t, window, g)
        assert np.all(r["cnt"] == 2) and np.all(r["flags"] == 0)
        np.testing.assert_allclose(r["twoF"], expect, rtol=1e-12)


def test_exp_window_large_tau_tends_to_rect():
    """I7: exp weights -> 1 as tau -> inf; the exp cell with 3 tau = L equals the rect cell
    of length L up to O(L/tau)."""
    t = (np.arange(6) * TSFT).astype(np.int32)
    atoms = make_atoms(t, np.random.default_rng(9)).astype(np.float32)
    tau = 600_000_000  # 3 tau fits int64 in the oracle; weights within 2e-5 of 1
    re = oracle.map2F(atoms, t, EXP, Grid(0, 1800, 2, tau, 1, 1))
    rr = oracle.map2F(atoms, t, RECT, Grid(0, 1800, 2, 6 * TSFT, 1, 1))
    assert np.array_equal(re["cnt"], rr["cnt"])
    np.testing.assert_allclose(re["twoF"], rr["twoF"], rtol=2e-4)
    assert not np.array_equal(re["twoF"], rr["twoF"])


def test_w_enters_linearly_on_F_and_quadratically_on_M():
    """With w on Fa,Fb and w^2 on a2,b2,ab a noise-free exp-injected signal is recovered with
    2F = rho^2 (test_injection_closed_form); here: a uniform rescale of a whole exp window by
    moving t0 one step earlier *without new atoms* must leave 2F unchanged (I3), which holds
    only for the (w, w^2) assignment."""
    t = np.array([7200, 9000, 10800, 12600], dtype=np.int32)
    atoms = make_atoms(t, np.random.default_rng(17)).astype(np.float32)
    tau = 50000
    r = oracle.map2F(atoms, t, EXP, Grid(3600, 3600, 2, tau, 1, 1))  # t0 = 3600, 7200
    assert r["cnt"].ravel().tolist() == [4, 4]
    np.testing.assert_allclose(r["twoF"][0, 0], r["twoF"][1, 0], rtol=1e-12)


# ----------------------------------------------------------------------------------------
# I9 noise-only statistics: 2F ~ chi^2 with 4 dof
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("window", [RECT, EXP])
def test_noise_only_chi2_4(window):
    """Across independent noise realisations at a FIXED well-conditioned cell (cells of one
    map are correlated, so a KS test over one map is invalid -- SURVEY.md 8(c) item 1)."""
    t = (np.arange(12) * TSFT).astype(np.int32)
    grid = Grid(1800, 1800, 1, 4 * 1800, 1800, 1)
    rng = np.random.default_rng(2024)
    vals = np.empty(4000)
    for i in range(vals.size):
        atoms = make_atoms(t, rng).astype(np.float32)
        r = oracle.map2F(atoms, t, window, grid, n_threads=1)
        assert r["flags"][0, 0] == 0
        vals[i] = r["twoF"][0, 0]
    assert abs(vals.mean() - 4.0) < 4 * np.sqrt(8.0 / vals.size)
    assert abs(vals.var() - 8.0) < 1.0
    assert stats.kstest(vals, "chi2", args=(4,)).pvalue > 1e-3


# ----------------------------------------------------------------------------------------
# marginalisation
# ----------------------------------------------------------------------------------------
def test_marginalise_against_scipy_and_bounds():
    rng = np.random.default_rng(4)
    m = rng.chisquare(4, size=(13, 29))
    fl = (rng.uniform(size=m.shape) < 0.2).astype(np.uint8)
    m[fl != 0] = 1e9  # must be ignored
    r = oracle.marginalise(m, fl)
    valid = m[fl == 0]
    assert r.n_valid == valid.size
    assert r.max2F == valid.max()
    flat = np.flatnonzero((m == valid.max()) & (fl == 0))[0]
    assert (r.m, r.n) == divmod(int(flat), m.shape[1])  # row-major, tau fastest
    assert abs(r.logB - logsumexp(0.5 * valid)) < 1e-12
    assert 0.5 * r.max2F <= r.logB <= 0.5 * r.max2F + np.log(r.n_valid)
    # constant map: logB = F + log n_valid
    c = np.full((5, 7), 6.0)
    rc = oracle.marginalise(c)
    assert abs(rc.logB - (3.0 + np.log(35))) < 1e-12 and (rc.m, rc.n) == (0, 0)
    # exact tie -> lowest flat index; large values do not overflow
    c[3, 2] = c[1, 4] = 4000.0
    rt = oracle.marginalise(c)
    assert (rt.m, rt.n) == (1, 4) and np.isfinite(rt.logB) and rt.logB > 2000.0


def test_search_equals_map_then_marginalise():
    grid = Grid(0, 1800, 8, 3600, 1800, 11)
    wl = tiny_workload(33, 40, 0.1, grid, n_templates=5, phi_random=True)
    res, terms = oracle.search(wl.data.atoms, wl.data.t, EXP, grid)
    tot = 0
    for k in range(5):
        r = oracle.map2F(wl.data.atoms[k], wl.data.t, EXP, grid)
        mg = oracle.marginalise(r["twoF"], r["flags"])
        assert (res[k].max2F, res[k].m, res[k].n, res[k].logB, res[k].n_valid) == (
            mg.max2F, mg.m, mg.n, mg.logB, mg.n_valid)
        tot += int(r["cnt"].sum())
    assert terms == tot
    assert len({(r.m, r.n) for r in res}) > 1  # templates really differ
