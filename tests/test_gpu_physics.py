"""Physics pins on the GPU at sizes no oracle reaches (statistical, loose by design; bit-exact
correctness is carried by the replay tests).  What the paper fixes:

* after a quench to T_c the energy approaches E_eq = -sqrt 2 monotonically from above
   with E(t) - E_eq ~ t^(-1/z), z = 2.1676(1) (Eq. 4 and 7);
* the coherence length grows as xi ~ t^(1/z) (Eq. 5).
"""
import math

import numpy as np
import pytest

import paper_2503_14688_b200 as lat
from paper_2503_14688_b200 import analysis
from paper_2503_14688_b200 import run as runner
from paper_2503_14688_b200 import workloads

pytestmark = pytest.mark.gpu
Z = 2.1676


def _slope(recs, key, t_lo, t_hi, shift=0.0):
    by_t = {r["t"]: r for r in recs}
    a, b = by_t[t_lo][key] + shift, by_t[t_hi][key] + shift
    return math.log(b / a) / math.log(t_hi / t_lo)


def test_config2_whole_run_energy_and_xi_scaling():
    """BASELINE.json config 2, whole: L = 4096, 20000 sweeps at beta_c, records at 2^k."""
    w = workloads.CONFIGS["ising_L4096"]
    recs = runner.run(w)
    ts = [r["t"] for r in recs]
    assert ts == w.measure_times() and ts[-1] == 20000
    e = np.array([r["e"] for r in recs])
    assert abs(e[0]) < 5e-3                                   # disordered start: e = 0 +- 2/L
    d = np.diff(e[1:])
    assert (d[np.array(ts[2:]) <= 4096] < 0).all()            # monotone decrease after the quench
    assert (d < 1e-3).all()                                   # later: up to the equilibrium noise ~ 1/L
    assert -math.sqrt(2) < e[-1] < -1.40                      # from above, close to -sqrt 2
    s_e = _slope(recs, "e", 64, 4096, shift=math.sqrt(2))
    assert abs(s_e + 1 / Z) < 0.06, s_e                       # E - E_eq ~ t^(-1/z)
    s_xi = _slope(recs, "xi", 256, 16384)
    assert 0.3 < s_xi < 0.6, s_xi                             # xi ~ t^(1/z), single-run estimator
    for r in recs:
        assert r["Q"] == w.L ** 2 and abs(r["m"]) < 0.05
        assert r["r_cut"] < w.r_max or r["t"] == 0            # the correlation sum was not truncated
    # C(r) decays: S(1) > S(8) > S(64) > 0 at the end of the run
    last = recs[-1]
    S = np.array(last["Sx"]) + np.array(last["Sy"])
    assert S[0] > S[7] > S[63] > 0


def test_checkpoint_resume_is_bit_identical(tmp_path):
    w = workloads.CONFIGS["bc_L2p15_ramp"]
    full = runner.run(w, sweeps=48, r_max=16, L=1024)
    runner.run(w, sweeps=32, r_max=16, L=1024)
    ck = str(tmp_path / "state.npz")
    runner.save_checkpoint(runner.run.last_lattice, ck)
    rest = runner.run(w, sweeps=48, r_max=16, resume=ck)
    strip = lambda r: {k: v for k, v in r.items() if k != "seconds_since_last_record"}
    assert [strip(r) for r in rest] == [strip(r) for r in full if r["t"] >= 32]


def test_config3_blume_capel_whole_run():
    """BASELINE.json config 3, whole (L = 16384, T = 1.6934, Delta = 0, 10000 sweeps, records at
    2^k): the energy decreases monotonically, vacancies thin out, no magnetisation develops,
    domains coarsen with xi ~ t^(1/z) (same universality class)."""
    w = workloads.CONFIGS["bc_L16384"]
    recs = runner.run(w, r_max=512)
    assert [r["t"] for r in recs] == w.measure_times() and recs[-1]["t"] == 10000
    e = np.array([r["e"] for r in recs])
    q = np.array([r["q"] for r in recs])
    assert abs(e[0]) < 2e-3 and abs(q[0] - 2 / 3) < 1e-3      # uniform on {-1, 0, +1}
    assert (np.diff(e) < 0).all() and (np.diff(q) > 0).all()
    assert q[-1] > 0.83 and e[-1] < -1.14
    assert all(abs(r["m"]) < 0.05 for r in recs)
    s_xi = _slope(recs, "xi", 256, 8192)
    assert 0.3 < s_xi < 0.6, s_xi                              # 1/z = 0.461
    assert all(r["r_cut"] < 512 for r in recs)


def test_dynamic_exponent_z_from_replicas_matches_the_paper():
    """The paper's headline number from its own procedure: 8 independent
    quenches of an L = 2^14 Ising lattice to T_c, C(r; t) at t = 2^k <= 4096, xi(t) = I_2/I_1 with the
    App. C cut-offs and tail fit, jackknife errors, and the fit of Eq. (5) with omega = 1.75.
    The paper finds z = 2.1676(1) (Eq. 7) with xi up to 1133; this short run reaches
    xi = 120 and must agree within its own (much larger) error."""
    w = workloads.CONFIGS["ising_L4096"]
    times, C, e = runner.replica_correlations(w, n_runs=8, sweeps=4096, r_max=1024, L=16384)
    fit = analysis.fit_z_jackknife(times, C, t_min=16)
    assert fit["dof"] == 6 and fit["Q"] > 0.1 and fit["chi2"] / fit["dof"] < 2.0, fit
    assert 0 < fit["z_err"] < 0.05
    assert abs(fit["z"] - Z) < max(3 * fit["z_err"], 0.05), fit
    xi = fit["xi"]
    assert (np.diff(xi) > 0).all() and 100 < xi[-1] < 140            # xi(4096) ~ 120
    # the energy route (Eq. 6) at leading order: E - E_eq ~ t^(-1/z)
    ex = np.array([x.mean() for x in e]) + math.sqrt(2)
    slope = math.log(ex[-1] / ex[6]) / math.log(times[-1] / times[6])
    assert abs(slope + 1 / Z) < 0.06


@pytest.mark.parametrize("name,e_plateau", [("ising_L2p16_ramp", -1.3583), ("bc_L2p15_ramp", -1.0993)])
def test_config5_protocol2_whole_runs(name, e_plateau):
    """BASELINE.json config 5, whole (20000 sweeps, beta ramps from 0.9 beta_f to beta_f = beta_c/1.01
    over the first 1000 sweeps, then constant): the energy follows the ramp down and then sits at
    the equilibrium value of T = 1.01 T_c -- above the critical -sqrt 2 for Ising -- while xi
    saturates at a finite value (the regime of PAPER.md:96, xi_eq(T_2) finite).  The plateau
    energies are this build's own numbers; what is asserted is that they are a plateau."""
    w = workloads.CONFIGS[name]
    recs = runner.run(w)
    by_t = {r["t"]: r for r in recs}
    assert sorted(by_t) == w.measure_times() and recs[-1]["t"] == 20000
    e = np.array([r["e"] for r in recs])
    assert (np.diff(e[:13]) < 0).all()                              # down the ramp (t <= 2048)
    late = np.array([by_t[t]["e"] for t in (4096, 8192, 16384, 20000)])
    assert np.ptp(late) < 1.5e-3 and abs(late.mean() - e_plateau) < 3e-3
    if w.model == lat.ISING:
        assert late.mean() > -math.sqrt(2) + 0.03                   # T > T_c: above E_eq(T_c)
    assert all(abs(r["m"]) < 0.01 for r in recs)
    assert 30 < by_t[20000]["xi"] < 250 and by_t[20000]["r_cut"] < w.r_max
