"""lattice_sweep_record: n sweeps + the r = 1 record, counted inside the last white half-sweep where that
kernel exists (Ising marching kernel, L > 4352), must return exactly what lattice_sweep followed by
lattice_measure(1) returns -- and leave exactly the same spins -- including the late tie flips that the
record has to be corrected for, beta = 0 (EDGE kernel), specialised and generic temperatures, and the
handles that fall back to the two separate calls."""
import math

import numpy as np
import pytest

import oracle
import paper_2503_14688_b200 as lat
from paper_2503_14688_b200 import workloads

pytestmark = pytest.mark.gpu
BETA_C = workloads.BETA_C_ISING


@pytest.mark.parametrize("scheme", [1, 2])
def test_fused_record_equals_sweep_then_measure_and_the_oracle(scheme):
    L, seed = 4608, 8086                           # marching kernel (not one row per thread)
    g = lat.Lattice(L, lat.ISING, 0.0, seed, scheme)
    s = lat.Lattice(L, lat.ISING, 0.0, seed, scheme)
    o = oracle.OracleLattice(L, lat.ISING, 0.0, seed, scheme)
    oracle.set_threads(16)
    # specialised beta_c, a generic beta, beta = 0 (every class "always": the EDGE kernel), low temperature
    for sched in ([BETA_C], [BETA_C] * 3, [0.3], [0.0], [BETA_C, 0.0, 1.0 / 1.66], [2.0], [BETA_C / 1.01] * 2):
        n0 = g.launches
        got = g.sweep_record(sched)
        assert g.launches - n0 <= 2 * len(sched)   # no measurement launch: the record rode on the last half-sweep
        s.sweep(sched)
        M, Q, Sx, Sy = s.measure(1)
        assert got == (M, Q, int(Sx[0]), int(Sy[0])), sched
        o.sweep(sched)
        Mo, Qo, Sxo, Syo = o.measure(1)
        assert got == (Mo, Qo, int(Sxo[0]), int(Syo[0])), sched
    assert np.array_equal(g.get_spins(), o.get_spins())
    assert g.time == s.time == o.time
    # ordered start: every lane needs a decision, ties (and late flips to correct for) are most frequent
    for d in (g, s):
        d.fill(1)
    for b in (BETA_C, 0.35, BETA_C):
        got = g.sweep_record([b])
        s.sweep([b])
        M, Q, Sx, Sy = s.measure(1)
        assert got == (M, Q, int(Sx[0]), int(Sy[0])), b
    assert np.array_equal(g.get_spins(), s.get_spins())
    # n = 0: the record of the state as it is
    M, Q, Sx, Sy = s.measure(1)
    assert g.sweep_record([]) == (M, Q, int(Sx[0]), int(Sy[0]))
    g.close(); s.close(); o.close()
    oracle.set_threads(1)


@pytest.mark.parametrize("model,L,delta", [(lat.ISING, 1024, 0.0), (lat.ISING, 192, 0.0), (lat.BLUME_CAPEL, 512, 0.0),
                                           (lat.BLUME_CAPEL, 256, 0.7)])
def test_record_falls_back_to_sweep_and_measure(model, L, delta):
    beta = BETA_C if model == lat.ISING else workloads.BETA_BC
    g = lat.Lattice(L, model, delta, 99)
    o = oracle.OracleLattice(L, model, delta, 99)
    for sched in ([beta] * 4, [beta, 0.0, beta]):
        got = g.sweep_record(sched)
        o.sweep(sched)
        Mo, Qo, Sxo, Syo = o.measure(1)
        assert got == (Mo, Qo, int(Sxo[0]), int(Syo[0]))
    assert np.array_equal(g.get_spins(), o.get_spins())
    with pytest.raises(lat.LatticeError):
        g.sweep_record([math.nan])
    g.close(); o.close()


def test_fused_record_at_full_size_against_the_one_pass_measurement():
    """L = 2^16 (the largest the whole-lattice comparison is cheap at): fused record = measure_e1 pass."""
    L = 1 << 16
    g = lat.Lattice(L, lat.ISING, 0.0, workloads.CONFIGS["ising_L2p16_ramp"].seed)
    for sched in ([BETA_C] * 2, [0.9 * BETA_C]):
        got = g.sweep_record(sched)
        M, Q, Sx, Sy = g.measure(1)
        assert got == (M, Q, int(Sx[0]), int(Sy[0]))
    g.close()
