"""Pins for the oracle's Metropolis dynamics (CPU only).

What the paper and the mathematics fix: the stationary law is Boltzmann (exact enumeration on
4x4 and 2x2), single-site flip frequencies equal thr/2^32 for the site's dE class, the
closed-form acceptance of the first half-sweep on an i.i.d. start, the T -> infinity and
T -> 0 limits, the Ising limit of Blume-Capel, and e(T_c) -> -sqrt(2) from
above after a quench.
"""
import math

import numpy as np
import pytest

import exact
import oracle

BETA_C = math.log(1 + math.sqrt(2)) / 2


def _series_stats(lat, n, beta, L, delta=0.0, burn=2000):
    lat.run_series(burn, beta)
    M, B, Q, _ = lat.run_series(n, beta)
    N = L * L
    e = (-B + delta * Q) / N
    return {
        "e": exact.binned_error(e),
        "abs_m": exact.binned_error(np.abs(M) / N),
        "m2": exact.binned_error((M / N) ** 2),
        "q": exact.binned_error(Q / N),
        "bond": exact.binned_error(-B / N),
    }


def _agree(stat, want, nsig=4.5):
    mean, err = stat
    assert abs(mean - want) < nsig * err + 1e-12, (mean, want, err)
    assert err < 0.01 * max(1.0, abs(want))           # the test has resolving power


@pytest.mark.parametrize("scheme,beta,n", [(0, BETA_C, 600_000), (1, BETA_C, 300_000),
                                           (0, 0.2, 400_000), (1, 0.6, 300_000)])
def test_ising_4x4_stationary_law(scheme, beta, n):
    ex = exact.ising_exact(4, beta)
    lat = oracle.OracleLattice(4, oracle.ISING, 0.0, seed=1234 + scheme, scheme=scheme)
    st = _series_stats(lat, n, beta, 4)
    _agree(st["e"], ex["e"])
    _agree(st["abs_m"], ex["abs_m"])
    _agree(st["m2"], ex["m2"])


@pytest.mark.parametrize("scheme,T,delta,n", [(0, 1.6934, 0.0, 600_000), (1, 1.6934, 0.0, 200_000),
                                              (0, 1.0, 1.0, 600_000), (1, 1.0, 1.0, 200_000)])
def test_blume_capel_4x4_stationary_law(scheme, T, delta, n):
    ex = exact.blume_capel_exact_4x4(1.0 / T, delta)
    lat = oracle.OracleLattice(4, oracle.BLUME_CAPEL, delta, seed=99 + scheme, scheme=scheme)
    st = _series_stats(lat, n, 1.0 / T, 4, delta)
    _agree(st["e"], ex["h"])
    _agree(st["bond"], ex["bond"])
    _agree(st["abs_m"], ex["abs_m"])
    _agree(st["q"], ex["q"])
    _agree(st["m2"], ex["m2"])


@pytest.mark.parametrize("model,values,beta,delta", [(oracle.ISING, (-1, 1), 0.3, 0.0),
                                                     (oracle.ISING, (-1, 1), 0.05, 0.0),
                                                     (oracle.BLUME_CAPEL, (-1, 0, 1), 0.4, 0.5)])
def test_2x2_state_histogram(model, values, beta, delta):
    """Empirical occupation of every state of the 2x2 lattice (bonds doubled by the wrap)
    against the exact law of the sweep chain started from the oracle's own initial state.

    The exact 16x16 (81x81) sweep matrix is built in tests/exact.py from the definition.  It
    leaves the Boltzmann law invariant (checked), but on 2x2 the Ising chain is not ergodic
    (dE = 0 moves are deterministic), so the long-run histogram is the Cesaro limit from the
    start state rather than Boltzmann itself -- which pins the dynamics even more sharply."""
    ex = exact.small_exact(2, values, beta, delta)
    P = exact.sweep_matrix(2, values, beta, delta)
    assert np.allclose(P.sum(axis=1), 1.0)
    assert np.allclose(ex["prob"] @ P, ex["prob"], atol=1e-12)       # pi P_black P_white = pi
    n = 400_000
    lat = oracle.OracleLattice(2, model, delta, seed=7, scheme=1)
    s0 = lat.get_spins().ravel().astype(int)
    q = len(values)
    start = sum(values.index(int(v)) * q ** x for x, v in enumerate(s0))
    want = exact.cesaro_limit(P, start)
    _, _, _, S = lat.run_series(n, beta, with_state=True)
    if q == 2:      # oracle codes are base 3 with digit sigma+1 in {0,2}; map to base 2
        digits = [(S // 3 ** x) % 3 // 2 for x in range(4)]
        S = sum(d * 2 ** x for x, d in enumerate(digits))
    nbins = 40
    per = n // nbins
    for k, pk in enumerate(want):
        occ = (S[: per * nbins] == k).reshape(nbins, per).mean(axis=1)
        mean, err = occ.mean(), occ.std(ddof=1) / math.sqrt(nbins)
        assert abs(mean - pk) < 5 * err + 3e-4, (k, mean, pk, err)
    if model == oracle.BLUME_CAPEL:
        assert np.allclose(want, ex["prob"], atol=1e-9)              # ergodic: Boltzmann itself


@pytest.mark.parametrize("scheme", [0, 1])
def test_single_site_flip_frequency_matches_threshold_class(scheme):
    """Fix a 4x4 configuration; over many seeds, a black half-sweep flips each black site with
    probability thr(dE)/2^32 where dE = 2*sigma*h is recomputed here from the definition."""
    rng = np.random.default_rng(5)
    x = rng.choice(np.array([-1, 1], dtype=np.int8), size=(4, 4))
    x[1, 1] = x[0, 1] = x[2, 1] = x[1, 0] = x[1, 2] = 1          # a k = 4 site
    x[2, 2], x[1, 2], x[3, 2], x[2, 3] = -1, 1, -1, -1            # (2,2): k = 3 (left is +1)
    n = 6000
    flips = np.zeros((4, 4))
    beta = BETA_C
    for seed in range(n):
        lat = oracle.OracleLattice.window(4, oracle.ISING, 0.0, seed, scheme, 3, 0, 0, x)
        lat.half_sweep(0, beta)
        flips += lat.get_spins() != x
    h = np.roll(x, 1, 0) + np.roll(x, -1, 0) + np.roll(x, 1, 1) + np.roll(x, -1, 1)
    dE = 2 * x.astype(int) * h
    for i in range(4):
        for j in range(4):
            f = flips[i, j] / n
            if (i + j) % 2 == 1:
                assert f == 0.0                                  # white untouched
                continue
            p = min(1.0, math.exp(-beta * dE[i, j]))
            assert abs(f - p) <= 4.5 * math.sqrt(p * (1 - p) / n) + 1e-12, (i, j, f, p)
    assert {4, 8} <= set(dE[::2, ::2].ravel()) | set(dE[1::2, 1::2].ravel())


def test_first_half_sweep_acceptance_closed_form_ising():
    # i.i.d. start: k ~ Binomial(4, 1/2) neighbours agree; accept = 11/16 + thr4/4 + thr8/16
    L = 1024
    r = math.sqrt(2) - 1
    want = 11 / 16 + r ** 2 / 4 + r ** 4 / 16
    assert abs(want - 0.7322330470336) < 1e-12
    for scheme in (0, 1):
        lat = oracle.OracleLattice(L, oracle.ISING, 0.0, seed=31 + scheme, scheme=scheme)
        before = lat.get_spins()
        lat.half_sweep(0, BETA_C)
        after = lat.get_spins()
        ii, jj = np.indices((L, L))
        black = (ii + jj) % 2 == 0
        assert (before[~black] == after[~black]).all()
        frac = (before[black] != after[black]).mean()
        nb = black.sum()
        assert abs(frac - want) < 4.5 * math.sqrt(want * (1 - want) / nb), (frac, want)


def test_first_half_sweep_acceptance_closed_form_blume_capel():
    L, T = 1024, 1.6934
    # average of min(1, exp(-beta dE)) over sigma uniform in 3, proposal fair, 4 iid neighbours
    want, cnt = 0.0, 0
    for s in (-1, 0, 1):
        for s2 in (-1, 0, 1):
            if s2 == s:
                continue
            for nb in np.ndindex(3, 3, 3, 3):
                h = sum(v - 1 for v in nb)
                dE = -(s2 - s) * h
                want += min(1.0, math.exp(-dE / T))
                cnt += 1
    want /= cnt
    assert abs(want - 0.7464822859015) < 1e-10
    lat = oracle.OracleLattice(L, oracle.BLUME_CAPEL, 0.0, seed=77, scheme=1)
    before = lat.get_spins()
    lat.half_sweep(0, 1 / T)
    after = lat.get_spins()
    ii, jj = np.indices((L, L))
    black = (ii + jj) % 2 == 0
    frac = (before[black] != after[black]).mean()
    assert abs(frac - want) < 4.5 * math.sqrt(want * (1 - want) / black.sum())


@pytest.mark.parametrize("scheme", [0, 1])
def test_infinite_temperature_limit(scheme):
    # beta = 0: thr = 2^32, every proposal accepted: Ising flips every spin each sweep
    lat = oracle.OracleLattice(32, oracle.ISING, 0.0, seed=3, scheme=scheme)
    s0 = lat.get_spins()
    M0, Q0, Sx0, Sy0 = lat.measure(8)
    lat.sweep([0.0])
    assert (lat.get_spins() == -s0).all()
    M1, Q1, Sx1, Sy1 = lat.measure(8)
    assert M1 == -M0 and (Sx1 == Sx0).all() and (Sy1 == Sy0).all()
    lat.sweep([0.0])
    assert (lat.get_spins() == s0).all()
    # Blume-Capel: every site changes value in its half-sweep, to the proposed value
    bc = oracle.OracleLattice(32, oracle.BLUME_CAPEL, 0.4, seed=3, scheme=scheme)
    b0 = bc.get_spins()
    bc.half_sweep(0, 0.0)
    b1 = bc.get_spins()
    ii, jj = np.indices((32, 32))
    black = (ii + jj) % 2 == 0
    assert (b1[black] != b0[black]).all() and (b1[~black] == b0[~black]).all()
    for i, j in [(0, 0), (5, 7), (30, 2)]:
        bit = oracle.proposal_bit(3, 0, 0, i * 16 + (j >> 1))
        assert b1[i, j] + 1 == (b0[i, j] + 1 + 1 + bit) % 3


@pytest.mark.parametrize("scheme", [0, 1])
def test_zero_temperature_limit(scheme):
    L = 32
    lat = oracle.OracleLattice(L, oracle.ISING, 0.0, seed=11, scheme=scheme)
    _, _, Sx, Sy = lat.measure(1)
    e_prev = -(Sx[0] + Sy[0])
    for _ in range(12):
        lat.sweep([math.inf])
        _, _, Sx, Sy = lat.measure(1)
        e = -(Sx[0] + Sy[0])
        assert e <= e_prev                      # thr = 0: the energy never increases
        e_prev = e
    up = np.ones((L, L), dtype=np.int8)
    lat2 = oracle.OracleLattice(L, oracle.ISING, 0.0, seed=12, scheme=scheme)
    lat2.set_spins(up)
    lat2.sweep([math.inf] * 2)
    assert (lat2.get_spins() == 1).all()        # fixed point
    # the all-up state is also a fixed point at any finite beta with probability ~1-thr8..., so
    # use beta = inf for the single overturned spin, which must flip back (dE = -8)
    for (i, j) in [(4, 4), (4, 5)]:
        up2 = up.copy()
        up2[i, j] = -1
        lat3 = oracle.OracleLattice(L, oracle.ISING, 0.0, seed=13, scheme=scheme)
        lat3.set_spins(up2)
        lat3.sweep([math.inf])
        assert (lat3.get_spins() == 1).all()


def test_blume_capel_ising_limit_delta_to_minus_infinity():
    """Delta -> -inf suppresses vacancies.  With Delta = -50, beta = 0.6 every
    move into sigma = 0 has dE >= 46 (thr = 0); a vacancy-free lattice stays vacancy-free and
    a +1 <-> -1 proposal is accepted with the Ising probability for dE = 2*sigma*h."""
    L, beta, delta = 64, 0.6, -50.0
    thr = oracle.thresholds(oracle.BLUME_CAPEL, delta, beta).reshape(3, 2, 9)
    ising = oracle.thresholds(oracle.ISING, 0.0, beta)
    assert (thr[2, 1] == 0).all() and (thr[0, 0] == 0).all()          # +-1 -> 0 never
    assert int(thr[2, 0, 4 + 2]) == int(ising[0]) and int(thr[2, 0, 4 + 4]) == int(ising[1])
    assert int(thr[0, 1, 4 - 2]) == int(ising[0]) and int(thr[0, 1, 4 - 4]) == int(ising[1])
    rng = np.random.default_rng(1)
    s = rng.choice(np.array([-1, 1], dtype=np.int8), size=(L, L))
    lat = oracle.OracleLattice(L, oracle.BLUME_CAPEL, delta, seed=5, scheme=1)
    lat.set_spins(s)
    lat.sweep([beta] * 20)
    out = lat.get_spins()
    assert (out != 0).all() and (out != s).any()
    # from a disordered start, vacancies die out quickly (0 -> +-1 has dE <= -46)
    lat2 = oracle.OracleLattice(L, oracle.BLUME_CAPEL, delta, seed=6, scheme=0)
    lat2.sweep([beta] * 8)
    assert (lat2.get_spins() != 0).all()


def test_quench_energy_approaches_minus_sqrt2_from_above():
    # after a quench to T_c, e(t) decreases towards -sqrt(2) from above
    L = 1024
    oracle.set_threads(8)
    try:
        lat = oracle.OracleLattice(L, oracle.ISING, 0.0, seed=2024, scheme=0)
        es = []
        for n in (1, 3, 12, 48, 192):                   # t = 1, 4, 16, 64, 256
            lat.sweep([BETA_C] * n)
            _, _, Sx, Sy = lat.measure(1)
            es.append(-(Sx[0] + Sy[0]) / L ** 2)
    finally:
        oracle.set_threads(1)
    assert all(a > b for a, b in zip(es, es[1:]))
    assert all(e > -math.sqrt(2) for e in es)
    assert es[-1] < -1.37
    # E - E_eq ~ t^(-1/z), z = 2.1676: slope -0.46 between t = 16 and 256;
    # at L = 1024 the statistical error of e is ~0.004, i.e. ~0.06 on the slope
    ex = [e + math.sqrt(2) for e in es]
    slope = math.log(ex[-1] / ex[2]) / math.log(256 / 16)
    assert -0.62 < slope < -0.32, slope


def test_window_replay_matches_full_lattice():
    """The windowed oracle (global keying, frozen outside) reproduces the inside of the full
    lattice as long as the dependency cone (2 sites per sweep) stays out of the inner block."""
    L, s = 64, 3
    for model, beta, out in [(oracle.ISING, BETA_C, 1), (oracle.BLUME_CAPEL, 0.59, 0)]:
        for scheme in (0, 1):
            full = oracle.OracleLattice(L, model, 0.0, seed=8, scheme=scheme)
            full.sweep([beta] * 5)
            i0, j0, h, w = 57, 60, 9, 11                     # wraps around both edges
            m = 2 * s
            win0 = full.get_spins((i0 - m) % L, (j0 - m) % L, h + 2 * m, w + 2 * m)
            win = oracle.OracleLattice.window(L, model, 0.0, 8, scheme, 5, (i0 - m) % L,
                                              (j0 - m) % L, win0, outside=out)
            betas = [beta * (1 + 0.01 * k) for k in range(s)]
            full.sweep(betas)
            win.sweep(betas)
            assert win.time == full.time == 8
            inner = win.get_spins(m, m, h, w)
            assert (inner == full.get_spins(i0, j0, h, w)).all()
            # and one more sweep lets the frozen boundary leak in somewhere (the test bites)
            whole = win.get_spins()
            ref = full.get_spins((i0 - m) % L, (j0 - m) % L, h + 2 * m, w + 2 * m)
            assert (whole != ref).any()
