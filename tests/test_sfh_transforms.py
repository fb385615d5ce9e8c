"""Host transforms of the paper's SFH models S1-S5 against closed forms."""
import numpy as np

from paper_1904_00011_b200 import sfh


def test_age_grid_midpoints_are_the_papers():
    m = sfh.age_midpoints(21)
    assert np.allclose(m[[0, 1, -1]], [6.1, 6.3, 10.1])


def test_every_model_sums_to_n_pix():
    for w in (sfh.ssp(9.3, 250.0), sfh.constant(250.0), sfh.tau_model(250.0, 3.0), sfh.tau_model(250.0, 3.0, delayed=True)):
        assert w.shape == (21,) and np.all(w >= 0) and abs(w.sum() - 250.0) < 1e-9
    assert np.count_nonzero(sfh.ssp(9.3, 250.0)) == 1 and sfh.ssp(9.3, 1.0)[16] == 1.0   # bin [9.2, 9.4)


def test_constant_sfr_is_proportional_to_linear_time():
    w = sfh.constant(1.0)
    e = 10.0 ** sfh.age_edges()
    assert np.allclose(w / w[0], (e[1:] - e[:-1]) / (e[1] - e[0]))
    assert np.allclose(w[1:] / w[:-1], 10 ** 0.2)                  # equal log bins: a constant ratio


def test_tau_models_limit_and_midpoint_rule():
    # tau -> infinity: exponential -> constant SFR; delayed -> SFR ~ t
    assert np.allclose(sfh.tau_model(1.0, 1e6), sfh.constant(1.0), rtol=1e-4)
    e = 10.0 ** sfh.age_edges()
    T = e[-1]
    w = sfh.tau_model(1.0, 1e6, delayed=True)
    want = ((T - e[:-1]) ** 2 - (T - e[1:]) ** 2)
    assert np.allclose(w, want / want.sum(), rtol=1e-4)
    # short tau: almost everything formed at the start (oldest bins)
    assert sfh.tau_model(1.0, 0.5)[-3:].sum() > 0.95
    # numerical quadrature of one bin
    tau = 2e9
    t = np.linspace(T - e[18], T - e[17], 20001)
    num = np.trapezoid(np.exp(-t / tau), t)
    all_t = np.linspace(0, T - e[0], 2000001)
    assert abs(sfh.tau_model(1.0, 2.0)[17] - num / np.trapezoid(np.exp(-all_t / tau), all_t)) < 1e-6


def test_non_parametric_spreads_at_constant_sfr_and_keeps_totals():
    edges = sfh.default_bins5()
    logs = np.array([0.5, 1.0, 1.5, 2.0, 1.2])
    w = sfh.non_parametric(logs, edges)
    assert abs(w.sum() - (10.0 ** logs).sum()) < 1e-9
    fe = sfh.age_edges()
    for k in range(5):                                             # coarse edges lie on fine edges
        sel = (fe[:-1] >= edges[k] - 1e-12) & (fe[1:] <= edges[k + 1] + 1e-12)
        assert abs(w[sel].sum() - 10.0 ** logs[k]) < 1e-9
        a = 10.0 ** fe
        rate = w[sel] / (a[1:] - a[:-1])[sel]
        assert np.allclose(rate, rate[0])                           # constant SFR inside a coarse bin
