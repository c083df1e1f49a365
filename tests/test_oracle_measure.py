"""Pins for the oracle's measurements and derived quantities (CPU only).

Brute-force double loops against identities that hold exactly:
parity of S(r), S(r) = S(L-r), sum_r S_x(r) = sum_i (row sum)^2, e from S(1) = direct bond
sum, uniform / Neel / striped states, and a closed form for the xi routine.
"""
import math

import numpy as np
import pytest

import oracle


def _random_lattice(L, model, seed):
    lat = oracle.OracleLattice(L, model, 0.3 if model else 0.0, seed=seed, scheme=1)
    lat.sweep([0.4] * 3)
    return lat


@pytest.mark.parametrize("model", [oracle.ISING, oracle.BLUME_CAPEL])
def test_measure_against_numpy_rolls(model):
    L = 24
    lat = _random_lattice(L, model, 4)
    s = lat.get_spins().astype(np.int64)
    M, Q, Sx, Sy = lat.measure(L - 1)
    assert M == s.sum() and Q == (s * s).sum()
    for r in range(1, L):
        assert Sx[r - 1] == (s * np.roll(s, -r, axis=1)).sum()
        assert Sy[r - 1] == (s * np.roll(s, -r, axis=0)).sum()


@pytest.mark.parametrize("model", [oracle.ISING, oracle.BLUME_CAPEL])
def test_measure_identities(model):
    L = 32
    lat = _random_lattice(L, model, 5)
    s = lat.get_spins().astype(np.int64)
    M, Q, Sx, Sy = lat.measure(L - 1)
    if model == oracle.ISING:
        assert Q == L * L
        assert all((int(v) - L * L) % 2 == 0 for v in np.concatenate([Sx, Sy]))
    for r in range(1, L):
        assert Sx[r - 1] == Sx[L - r - 1] and Sy[r - 1] == Sy[L - r - 1]
    # sum over all separations (r = 0 contributes Q) = sum of squared line sums
    assert Q + Sx.sum() == (s.sum(axis=1) ** 2).sum()
    assert Q + Sy.sum() == (s.sum(axis=0) ** 2).sum()
    # energy from S(1) equals the direct sum over bonds
    bonds = sum(int(s[i, j]) * int(s[i, (j + 1) % L]) + int(s[i, j]) * int(s[(i + 1) % L, j])
                for i in range(L) for j in range(L))
    delta = lat.delta
    e = oracle.energy(Sx, Sy, Q, delta, L)
    assert e == pytest.approx((-bonds + delta * Q) / L ** 2, rel=1e-15, abs=1e-15)


def test_measure_rows_partition_the_lattice():
    L = 32
    lat = _random_lattice(L, oracle.BLUME_CAPEL, 6)
    M, Q, Sx, Sy = lat.measure(9)
    parts = [lat.measure(9, rows=(i0, n)) for i0, n in [(0, 5), (5, 20), (25, 7)]]
    assert M == sum(p[0] for p in parts) and Q == sum(p[1] for p in parts)
    assert (Sx == sum(p[2] for p in parts)).all() and (Sy == sum(p[3] for p in parts)).all()
    s = lat.get_spins().astype(np.int64)
    # a slab's S_y pairs base rows i0..i0+n-1 with rows i+r (which may leave the slab)
    i0, n, r = 25, 7, 9
    assert parts[2][3][r - 1] == sum((s[i] * s[(i + r) % L]).sum() for i in range(i0, i0 + n))
    assert oracle.pair_sum(s[3], s[(3 + r) % L], 0) == (s[3] * s[(3 + r) % L]).sum()
    assert oracle.pair_sum(s[3], s[3], r) == (s[3] * np.roll(s[3], -r)).sum()


def test_special_states():
    L = 16
    lat = oracle.OracleLattice(L, oracle.ISING, 0.0, seed=1)
    ii, jj = np.indices((L, L))
    lat.set_spins(np.ones((L, L), dtype=np.int8))
    M, Q, Sx, Sy = lat.measure(L // 2)
    assert M == L * L and (Sx == L * L).all() and (Sy == L * L).all()
    lat.set_spins((1 - 2 * ((ii + jj) % 2)).astype(np.int8))            # Neel
    M, Q, Sx, Sy = lat.measure(L // 2)
    sign = np.array([(-1) ** r for r in range(1, L // 2 + 1)])
    assert M == 0 and (Sx == sign * L * L).all() and (Sy == sign * L * L).all()
    lat.set_spins((1 - 2 * (jj % 2)).astype(np.int8))                   # stripes along columns
    M, Q, Sx, Sy = lat.measure(L // 2)
    assert (Sx == sign * L * L).all() and (Sy == L * L).all()
    lat.set_spins((1 - 2 * (ii % 2)).astype(np.int8))                   # stripes along rows
    M, Q, Sx, Sy = lat.measure(L // 2)
    assert (Sy == sign * L * L).all() and (Sx == L * L).all()
    xi, rc = oracle.xi(Sx, Sy, Q, L)
    assert (xi, rc) == (0.0, 0)               # Sx(1) + Sy(1) = L^2 - L^2 = 0: cut at once
    # a direction-dependent pattern: period 4 along x only
    lat.set_spins(np.where(jj % 4 < 2, 1, -1).astype(np.int8))
    M, Q, Sx, Sy = lat.measure(4)
    assert list(Sx) == [0, -L * L, 0, L * L] and (Sy == L * L).all()


def test_xi_closed_form_geometric_correlations():
    # S(r) ~ x^r: sum r^2 x^r / sum r x^r = (1+x)/(1-x) = coth(1/(2a)) for x = exp(-1/a)
    for a, want in [(5.0, 10.0333111), (50.0, 100.003333311)]:
        x = math.exp(-1.0 / a)
        r_max = int(60 * a)
        amp = 2.0 ** 61
        S = np.array([int(amp * x ** r) for r in range(1, r_max + 1)], dtype=np.int64)
        S = np.maximum(S, 1)
        xi, rc = oracle.xi(S, S, Q=123, L=1 << 20)
        assert rc == r_max
        assert xi == pytest.approx((1 + x) / (1 - x), rel=2e-9)
        assert xi == pytest.approx(want, rel=1e-8)


def test_xi_cutoff_rule_and_weights():
    # r_cut = (first r with Sx+Sy <= 0) - 1; trapezoid: half weight at r_cut
    Sx = np.array([10, 6, 3, -1, 5, 5], dtype=np.int64)
    Sy = np.array([10, 6, 3, 1, 5, 5], dtype=np.int64)           # sum at r=4 is 0 -> r_cut = 3
    xi, rc = oracle.xi(Sx, Sy, Q=0, L=8)
    assert rc == 3
    C = np.array([20, 12, 6]) / (2 * 64)
    I1 = 1 * C[0] + 2 * C[1] + 0.5 * 3 * C[2]
    I2 = 1 * C[0] + 4 * C[1] + 0.5 * 9 * C[2]
    assert xi == pytest.approx(I2 / I1, rel=1e-15)
    xi0, rc0 = oracle.xi(np.array([-1], dtype=np.int64), np.array([0], dtype=np.int64), 0, 8)
    assert (xi0, rc0) == (0.0, 0)
    xi1, rc1 = oracle.xi(np.array([3, -9], dtype=np.int64), np.array([3, 0], dtype=np.int64), 0, 8)
    assert rc1 == 1 and xi1 == pytest.approx(1.0)


def test_argument_validation():
    lat = oracle.OracleLattice(8, oracle.ISING, 0.0, seed=1)
    with pytest.raises(oracle.OracleError):
        lat.measure(8)                       # r_max <= L-1
    with pytest.raises(oracle.OracleError):
        lat.sweep([-0.1])
    with pytest.raises(oracle.OracleError):
        lat.sweep([float("nan")])
    with pytest.raises(oracle.OracleError):
        lat.set_spins(np.zeros((2, 2), dtype=np.int8))          # 0 is not an Ising spin
    lat.sweep([0.4])
    assert lat.time == 1
    assert oracle.lib().oracle_set_rng_scheme(lat._h, 0) == oracle.ESTATE
    with pytest.raises(oracle.OracleError):
        oracle.OracleLattice(7, oracle.ISING, 0.0, seed=1)      # odd L
