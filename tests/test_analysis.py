"""The estimator layer (paper_2503_14688_b200/analysis.py) on synthetic data with known answers."""
import math

import numpy as np
import pytest

from paper_2503_14688_b200 import analysis as an


def test_jackknife_reduces_to_the_standard_error_for_the_mean():
    rng = np.random.default_rng(1)
    x = rng.normal(3.0, 2.0, size=(50, 4))
    mean, err = an.jackknife(x)
    assert np.allclose(mean, x.mean(axis=0))
    assert np.allclose(err, x.std(axis=0, ddof=1) / math.sqrt(50))
    # a nonlinear estimator: error of the square of the mean ~ 2 |mean| sigma_mean
    sq, sq_err = an.jackknife(x[:, 0], lambda m: m ** 2)
    assert abs(sq_err / (2 * abs(x[:, 0].mean()) * x[:, 0].std(ddof=1) / math.sqrt(50)) - 1) < 0.05
    with pytest.raises(ValueError):
        an.jackknife(x[:1])


def _synthetic_C(xiF, beta, R, A=1.0):
    r = np.arange(R + 1, dtype=np.float64)
    C = np.ones(R + 1)
    C[1:] = A * np.exp(-(r[1:] / xiF) ** beta) / np.sqrt(r[1:])
    return C


@pytest.mark.parametrize("xiF,beta", [(20.0, 1.0), (35.0, 1.4), (12.0, 0.8)])
def test_xi_appendix_c_recovers_the_tail_function(xiF, beta):
    """For C(r) = A exp[-(r/xi_F)^beta] / sqrt(r) (Eq. C2), I_n = A xi_F^(n+1/2) Gamma((n+1/2)/beta)/beta,
    so xi = I_2/I_1 = xi_F Gamma(2.5/beta) / Gamma(1.5/beta)."""
    R = 2000
    C = _synthetic_C(xiF, beta, R, A=0.7)
    err = np.full(R + 1, 1e-9)
    d = {}
    xi = an.xi_appendix_c(C, err, d)
    exact = xiF * math.gamma(2.5 / beta) / math.gamma(1.5 / beta)
    assert abs(xi / exact - 1) < 0.02, (xi, exact, d)
    assert d["tail_fit"] and d["r_star"] < d["r_min"] < d["r_max"] < d["r_cut"]
    assert abs(d["xi_F"] / xiF - 1) < 1e-3 and abs(d["beta"] - beta) < 1e-3
    # with large errors the cut-off comes early and the data are integrated as they are
    d2 = {}
    with pytest.warns(an.CutoffWarning):
        an.xi_appendix_c(C, np.full(R + 1, 0.05), d2)
    assert d2["r_cut"] < d["r_cut"] and C[d2["r_cut"] + 1] < 0.15 <= C[d2["r_cut"]]


def test_xi_appendix_c_flags_missing_cutoffs():
    """r_max (r^2 C below a third of its maximum) does not occur inside the measured range: the
    routine integrates up to r_cut only, says so in details and warns; strict=True raises."""
    C = _synthetic_C(400.0, 1.0, 300)                    # r^2 C still rising at r = 300
    err = np.full(C.size, 1e-9)
    d = {}
    with pytest.warns(an.CutoffWarning):
        xi = an.xi_appendix_c(C, err, d)
    assert d["condition_met"] is False and d["r_max"] is None and not d["tail_fit"]
    exact = 400.0 * math.gamma(2.5) / math.gamma(1.5)
    assert xi < 0.5 * exact                              # the truncation bias the warning is about
    with pytest.raises(ValueError):
        an.xi_appendix_c(C, err, strict=True)
    d2 = {}
    an.xi_appendix_c(_synthetic_C(20.0, 1.0, 2000), np.full(2001, 1e-9), d2)
    assert d2["condition_met"] is True


def test_xi_with_error_freezes_the_cutoffs_of_the_full_sample():
    rng = np.random.default_rng(5)
    C = _synthetic_C(25.0, 1.2, 800)
    runs = C[None, :] + rng.normal(0.0, 2e-4, size=(20, C.size))
    d = {}
    an.xi_with_error(runs, d)
    seen = []
    orig = an.xi_appendix_c

    def spy(C_, E_, details=None, cutoffs=None, strict=False):
        seen.append(cutoffs)
        return orig(C_, E_, details, cutoffs, strict)

    an.xi_appendix_c = spy
    try:
        an.xi_with_error(runs)
    finally:
        an.xi_appendix_c = orig
    frozen = [c for c in seen if c is not None]
    assert len(frozen) == 21                                         # full mean + 20 leave-one-out
    assert all(c["r_cut"] == d["r_cut"] and c["r_min"] == d["r_min"] and c["r_max"] == d["r_max"] for c in frozen)


def test_xi_with_error_on_noisy_runs():
    rng = np.random.default_rng(7)
    C = _synthetic_C(25.0, 1.2, 800)
    runs = C[None, :] + rng.normal(0.0, 2e-4, size=(40, C.size))
    xi, err = an.xi_with_error(runs)
    exact = 25.0 * math.gamma(2.5 / 1.2) / math.gamma(1.5 / 1.2)
    assert 0 < err < 0.05 * exact and abs(xi - exact) < max(5 * err, 0.03 * exact)


def test_fit_z_recovers_the_exponent_of_eq_5():
    """Points generated from log t = z log xi + b + b' xi^-omega are fitted back exactly."""
    z, b, b1 = 2.1676, -0.35, 1.9
    xi = np.geomspace(5.0, 1100.0, 18)
    t = np.exp(z * np.log(xi) + b + b1 * xi ** (-an.OMEGA))
    fit = an.fit_z(t, xi, 1e-3 * xi)
    assert abs(fit["z"] - z) < 1e-9 and abs(fit["b"] - b) < 1e-8 and abs(fit["b1"] - b1) < 1e-6
    assert fit["dof"] == 15 and fit["chi2"] < 1e-12 and fit["Q"] > 0.999
    # t_min drops the early points; too few points is an error
    assert an.fit_z(t, xi, 1e-3 * xi, t_min=t[10])["dof"] == 5
    with pytest.raises(ValueError):
        an.fit_z(t, xi, 1e-3 * xi, t_min=t[-3])
    # noisy xi: z within a few sigma of chi^2-consistent noise, Q not tiny
    rng = np.random.default_rng(3)
    noisy = xi * (1 + 2e-3 * rng.normal(size=xi.size))
    f2 = an.fit_z(t, noisy, 2e-3 * xi)
    assert abs(f2["z"] - z) < 0.02 and f2["Q"] > 1e-3


def test_fit_z_jackknife_on_synthetic_runs():
    rng = np.random.default_rng(11)
    z, b, b1 = 2.1676, 0.1, 1.0
    xiF = np.geomspace(6.0, 60.0, 8)
    ratio = math.gamma(2.5 / 1.3) / math.gamma(1.5 / 1.3)
    xi_true = xiF * ratio
    t = np.exp(z * np.log(xi_true) + b + b1 * xi_true ** (-an.OMEGA))
    stacks = [_synthetic_C(x, 1.3, 1200)[None, :] + rng.normal(0, 1e-5, size=(12, 1201)) for x in xiF]
    fit = an.fit_z_jackknife(t, stacks)
    assert abs(fit["z"] - z) < 0.05 and 0 <= fit["z_err"] < 0.05
    assert np.all(np.abs(fit["xi"] / xi_true - 1) < 0.02)


def test_fit_z_energy_recovers_eq_6():
    """Points generated from Eq. (6) / (D2) are fitted back: z and the three amplitudes."""
    z, b, b1, b2 = 2.1676, 0.31, -0.12, 0.4
    t = np.geomspace(16, 524288, 40)
    E = an.E_EQ_ISING + b * t ** (-1 / z) + b1 * t ** (-2 / z) + b2 * t ** (-(an.OMEGA + 1.0) / z)
    fit = an.fit_z_energy(t, E, np.full(t.size, 1e-9))
    assert abs(fit["z"] - z) < 1e-6 and abs(fit["b"] - b) < 1e-5 and fit["dof"] == 36 and fit["chi2"] < 1.0
    assert an.fit_z_energy(t, E, np.full(t.size, 1e-9), t_min=1000.0)["dof"] < 36
    rng = np.random.default_rng(2)
    noisy = E + 2e-6 * rng.normal(size=t.size)
    f2 = an.fit_z_energy(t, noisy, np.full(t.size, 2e-6))
    assert abs(f2["z"] - z) < 0.02 and f2["Q"] > 1e-3
    with pytest.raises(ValueError):
        an.fit_z_energy(t[:4], E[:4], np.full(4, 1e-9))
    # a wrong E_eq is not absorbed: the fit quality collapses (why the paper uses it for Ising only)
    bad = an.fit_z_energy(t, noisy, np.full(t.size, 2e-6), E_eq=an.E_EQ_ISING + 1e-3)
    assert bad["chi2"] > 10 * f2["chi2"]


def test_fit_z_joint_shares_one_exponent_across_data_sets():
    """xi (Eq. 5) of two 'models' with different amplitudes + E (Eq. 6): one z for all (Fig. 3)."""
    z = 2.1676
    rng = np.random.default_rng(4)
    sets = []
    for b, b1 in ((-0.35, 1.9), (0.4, -0.8)):
        xi = np.geomspace(6.0, 1100.0, 16)
        t = np.exp(z * np.log(xi) + b + b1 * xi ** (-an.OMEGA))
        sets.append({"kind": "xi", "t": t, "xi": xi * (1 + 1e-4 * rng.normal(size=xi.size)), "xi_err": 1e-4 * xi})
    tE = np.geomspace(32, 524288, 24)
    E = an.E_EQ_ISING + 0.3 * tE ** (-1 / z) - 0.1 * tE ** (-2 / z) + 0.2 * tE ** (-(an.OMEGA + 1.0) / z)
    sets.append({"kind": "E", "t": tE, "E": E + 1e-7 * rng.normal(size=tE.size), "E_err": np.full(tE.size, 1e-7)})
    fit = an.fit_z_joint(sets)
    assert abs(fit["z"] - z) < 2e-3 and fit["dof"] == 16 + 16 + 24 - (1 + 2 + 2 + 3)
    assert fit["Q"] > 1e-3 and len(fit["amplitudes"]) == 3
    assert abs(fit["amplitudes"][0][0] + 0.35) < 0.02 and abs(fit["amplitudes"][2][0] - 0.3) < 0.01
    single = an.fit_z_joint(sets[:1])                     # one xi set: the same answer as fit_z
    ref = an.fit_z(sets[0]["t"], sets[0]["xi"], sets[0]["xi_err"])
    assert abs(single["z"] - ref["z"]) < 1e-6


def test_fit_z_energy_jackknife_and_exponential_approach():
    rng = np.random.default_rng(9)
    z = 2.17
    t = np.geomspace(64, 262144, 20)
    E = an.E_EQ_ISING + 0.3 * t ** (-1 / z) - 0.05 * t ** (-2 / z)
    runs = [E[k] + 3e-6 * rng.normal(size=24) for k in range(t.size)]
    fit = an.fit_z_energy_jackknife(t, runs)
    assert abs(fit["z"] - z) < 0.05 and 0 < fit["z_err"] < 0.05
    # Eq. (8): one tau for all f, b(f) changes sign around f = 0.59
    tau = 3.0e4
    tt = np.linspace(4e4, 3e5, 30)
    curves = [{"f": f, "t": tt, "E": an.E_EQ_ISING + b * np.exp(-tt / tau) + 1e-8 * rng.normal(size=tt.size),
               "E_err": np.full(tt.size, 1e-8)} for f, b in ((0.54, 1.5e-4), (0.59, 0.0), (0.64, -2.4e-4))]
    res = an.fit_exponential_approach(curves)
    assert abs(res["tau"] / tau - 1) < 0.01
    assert abs(res["b"][0.54] - 1.5e-4) < 2e-6 and abs(res["b"][0.59]) < 2e-6 and res["b"][0.64] < -2e-4
    free = an.fit_exponential_approach(curves, E_eq=None)            # Blume-Capel: E_eq is a parameter
    assert abs(free["E_eq"] - an.E_EQ_ISING) < 1e-7 and abs(free["tau"] / tau - 1) < 0.02


def test_sparse_r_grid_spline_reproduces_the_dense_estimate():
    """C(r) sampled on a log-spaced r-grid and splined gives the dense-grid xi."""
    C = _synthetic_C(30.0, 1.3, 1500, A=0.8)
    err = np.full(C.size, 1e-9)
    dense = an.xi_appendix_c(C, err)
    r = np.unique(np.round(np.geomspace(1, 1500, 90)).astype(int))
    sparse = an.xi_sparse(r, C[r], err[r])
    assert abs(sparse / dense - 1) < 5e-3
    d, e = an.densify(r, C[r], err[r])
    assert d.size == 1501 and np.allclose(d[r], C[r]) and e.size == 1501
    with pytest.raises(ValueError):
        an.densify([3, 2], [0.1, 0.2])
