"""Host logic of the Appendix-A timing-model fit (paper_1805_05652_b200/timing_model.py): times
manufactured from known constants must give those constants back."""
import numpy as np

from paper_1805_05652_b200.timing_model import fit, setups


def test_three_step_fit_recovers_known_constants():
    true = dict(c_call=2.0e-5, c_SFTs=3.0e-10, c_sums_r=2.0e-12, c_F=4.0e-12, c_sums_e=2.8e-13)
    rng = np.random.default_rng(0)
    rows = []
    for name, n_sft, g in setups(365.0, False):
        cells = g.N_t0 * g.N_tau
        # eqs. (A.5), (A.6) on gapless data, dt0 = dtau = T_SFT (half-open windows)
        m = np.arange(g.N_t0)[:, None] * (g.dt0 // 1800)
        n = (g.tau_min + np.arange(g.N_tau)[None, :] * g.dtau) // 1800
        for wname, k, c in (("rect", 1, true["c_sums_r"]), ("exp", 3, true["c_sums_e"])):
            n_sums = int(np.minimum(np.maximum(n_sft - m, 0), k * n).sum())
            sec = (true["c_call"] + true["c_SFTs"] * n_sft + c * n_sums + true["c_F"] * cells)
            rows.append(dict(setup=name, window=wname, n_sft=n_sft, N_t0=g.N_t0, N_tau=g.N_tau,
                             cells=cells, n_sums=n_sums,
                             seconds=sec * (1.0 + 0.002 * rng.standard_normal())))
    f = fit(rows)
    assert abs(f["c_call"] - true["c_call"]) / true["c_call"] < 0.05
    assert abs(f["c_sums_e"] - true["c_sums_e"]) / true["c_sums_e"] < 0.02
    assert abs((f["c_sums_r"] + f["c_F"]) - (true["c_sums_r"] + true["c_F"])) < 0.2 * 6e-12
    assert abs(f["c_e_PGM"] - 3 * true["c_sums_e"]) / (3 * true["c_sums_e"]) < 0.02
    assert f["median_relative_residual"]["exp"] < 0.01
