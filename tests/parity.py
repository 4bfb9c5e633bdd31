"""Shared comparison helpers for the GPU parity tests (tolerances of BASELINE.json north_star).

  |d 2F| <= 1e-3 * max(1, 2F)   on cells with oracle cond = D/(AB) >= 1e-6
  identical degenerate-cell flags (bit 0 always; bit 1 where cond >= 1e-6)
  logB within 1e-4 * max(1, |logB|)
  exact argmax unless the top two oracle values tie within the 2F tolerance
"""
import numpy as np

TOL_2F = 1e-3
TOL_LOGB = 1e-4
COND_MIN = 1e-6


def check_cells(g2F, gflags, ref, what=""):
    """g2F/gflags: GPU values (any shape); ref: dict from oracle.map2F / oracle.cells."""
    g2F = np.asarray(g2F, dtype=np.float64).ravel()
    r2F = ref["twoF"].ravel()
    rfl = ref["flags"].ravel()
    cond = ref["cond"].ravel()
    well = (cond >= COND_MIN) | ((rfl & 1) != 0)  # count-degenerate cells are always decidable
    if gflags is not None:
        gfl = np.asarray(gflags).ravel()
        assert np.array_equal(gfl & 1, rfl & 1), f"{what}: min_atoms flag differs"
        assert np.array_equal(gfl[well], rfl[well]), f"{what}: D<=0 flag differs"
        valid = (gfl == 0) & (rfl == 0)
    else:
        valid = rfl == 0
    chk = valid & (cond >= COND_MIN)
    err = np.abs(g2F - r2F)
    tol = TOL_2F * np.maximum(1.0, r2F)
    bad = chk & ~(err <= tol)
    assert not bad.any(), (f"{what}: {bad.sum()} cells outside tolerance, worst "
                           f"{(err / tol)[chk].max():.3g} x tol")
    assert np.all(g2F[rfl != 0][well[rfl != 0]] == 0.0), f"{what}: degenerate cell not stored as 0"
    return float((err / tol)[chk].max()) if chk.any() else 0.0


def check_result(got, ref_map, ref_flags, N_tau, what=""):
    """got: one RESULT_DTYPE record; ref_map/flags: the oracle's full fp64 map."""
    import oracle

    mg = oracle.marginalise(ref_map, ref_flags)
    assert int(got["n_valid"]) == mg.n_valid, f"{what}: n_valid {got['n_valid']} != {mg.n_valid}"
    if mg.n_valid == 0:
        assert (got["m"], got["n"], got["max2F"]) == (-1, -1, 0.0) and got["logB"] == -np.inf
        return
    assert abs(got["max2F"] - mg.max2F) <= TOL_2F * max(1.0, mg.max2F), f"{what}: max2F"
    assert abs(got["logB"] - mg.logB) <= TOL_LOGB * max(1.0, abs(mg.logB)), (
        f"{what}: logB {got['logB']} vs {mg.logB}")
    if (int(got["m"]), int(got["n"])) != (mg.m, mg.n):
        # allowed only if the oracle's value at the GPU's argmax ties with its maximum
        v = ref_map[int(got["m"]), int(got["n"])]
        assert ref_flags[int(got["m"]), int(got["n"])] == 0
        assert mg.max2F - v <= TOL_2F * max(1.0, mg.max2F), (
            f"{what}: argmax ({got['m']},{got['n']}) vs ({mg.m},{mg.n}) not a tie")
