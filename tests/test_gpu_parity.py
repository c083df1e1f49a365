"""GPU parity: the CUDA path, called through the C ABI, against the CPU oracle on the same
seeded inputs.  Spins and integer counts must match bit for bit; xi to 1e-12 relative
(BASELINE.json north_star)."""
import math
import os

import numpy as np
import pytest

import oracle
import paper_2503_14688_b200 as lat
from paper_2503_14688_b200 import workloads

pytestmark = pytest.mark.gpu

BETA_C = workloads.BETA_C_ISING
NCPU = os.cpu_count() or 1


@pytest.fixture(autouse=True)
def _threads():
    oracle.set_threads(NCPU)
    yield
    oracle.set_threads(1)


def _same_measure(g, o, r_max, L, delta=0.0, rows=None):
    Mg, Qg, Sxg, Syg = g.measure(r_max, rows)
    Mo, Qo, Sxo, Syo = o.measure(r_max, rows)
    assert (Mg, Qg) == (Mo, Qo)
    assert np.array_equal(Sxg, Sxo) and np.array_equal(Syg, Syo)
    if rows is None:
        xg, rg = lat.xi(Sxg, Syg, Qg, L)
        xo, ro = oracle.xi(Sxo, Syo, Qo, L)
        assert rg == ro
        assert xg == xo or abs(xg - xo) <= 1e-12 * abs(xo)          # north_star tolerance
        eg, eo = lat.energy(Sxg, Syg, Qg, delta, L), oracle.energy(Sxo, Syo, Qo, delta, L)
        assert eg == eo or abs(eg - eo) <= 1e-12 * abs(eo)


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
@pytest.mark.parametrize("L", [64, 128, 192, 256, 768, 1024])
def test_initial_state(L, model):
    g = lat.Lattice(L, model, 0.0, seed=77 + L)
    o = oracle.OracleLattice(L, model, 0.0, seed=77 + L)
    assert np.array_equal(g.get_spins(), o.get_spins())
    _same_measure(g, o, min(L // 2, 48), L)


@pytest.mark.parametrize("scheme", [0, 1])
def test_config1_ising_L64_whole_run(scheme):
    """BASELINE.json config 1, whole: 2000 sweeps at beta_c, records at sweeps 2^k."""
    w = workloads.CONFIGS["ising_L64"]
    g = lat.Lattice(w.L, w.model, w.delta, w.seed, scheme)
    o = oracle.OracleLattice(w.L, w.model, w.delta, w.seed, scheme)
    done = 0
    for t in w.measure_times():
        beta = w.beta_schedule(t - done, done)
        if t > done:
            g.sweep(beta)
            o.sweep(beta)
            done = t
        assert g.time == o.time == t
        assert np.array_equal(g.get_spins(), o.get_spins()), t
        _same_measure(g, o, w.r_max, w.L)


@pytest.mark.parametrize("scheme", [0, 1])
@pytest.mark.parametrize("L,sweeps", [(128, 300), (192, 100), (256, 200), (512, 100), (768, 40),
                                      (2048, 24)])
def test_ising_sweeps(L, sweeps, scheme):
    g = lat.Lattice(L, lat.ISING, 0.0, 4242 + L, scheme)
    o = oracle.OracleLattice(L, lat.ISING, 0.0, 4242 + L, scheme)
    for n in (1, 1, sweeps - 2):
        g.sweep([BETA_C] * n)
        o.sweep([BETA_C] * n)
        assert np.array_equal(g.get_spins(), o.get_spins())
    _same_measure(g, o, min(L // 2, 64), L)


@pytest.mark.parametrize("scheme", [0, 1])
@pytest.mark.parametrize("L,delta,T,sweeps", [(64, 0.0, 1.6934, 400), (128, 0.0, 1.6934, 100),
                                              (192, 0.7, 1.2, 60), (256, 0.0, 1.6934, 100),
                                              (256, -1.3, 2.0, 60), (512, 1.965, 0.6, 40),
                                              (1024, 0.0, 1.6934, 24), (256, -50.0, 1.5, 30)])
def test_blume_capel_sweeps(L, delta, T, sweeps, scheme):
    g = lat.Lattice(L, lat.BLUME_CAPEL, delta, 31 + L, scheme)
    o = oracle.OracleLattice(L, lat.BLUME_CAPEL, delta, 31 + L, scheme)
    for n in (1, 1, sweeps - 2):
        g.sweep([1.0 / T] * n)
        o.sweep([1.0 / T] * n)
        assert np.array_equal(g.get_spins(), o.get_spins())
    _same_measure(g, o, min(L // 2, 64), L, delta)


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
@pytest.mark.parametrize("scheme", [0, 1])
def test_half_sweeps_and_extreme_temperatures(model, scheme):
    L = 256
    g = lat.Lattice(L, model, 0.3, 5, scheme)
    o = oracle.OracleLattice(L, model, 0.3, 5, scheme)
    for beta in (0.0, 0.0, math.inf, 1e-12, 40.0, 0.3, math.inf, 0.0):
        for colour in (0, 1):
            g.half_sweep(colour, beta)
            o.half_sweep(colour, beta)
            assert np.array_equal(g.get_spins(), o.get_spins()), (beta, colour)
        g.sweep([beta])
        o.sweep([beta])
        assert np.array_equal(g.get_spins(), o.get_spins()), beta


@pytest.mark.parametrize("scheme", [1, 2])
def test_blume_capel_table_specialised_kernels_are_bit_identical(scheme):
    """The Blume-Capel counterpart: truth tables compiled in for T = 1.6934 / T_c / T_2 (one set), the
    plateau of config 5b's ramp and T_1 = 1.24 of the two-step protocol (Table II);
    any other beta, and any Delta != 0, takes the dispatching kernel."""
    from paper_2503_14688_b200 import workloads
    sp = lat.lib().lattice_plane_case_specialised
    specials = [workloads.BETA_BC, 1.0 / 1.69355839821214427017, 1.0 / 1.69661396797728, workloads.BETA_BC / 1.01,
                1.0 / 1.24]
    for b in specials:
        assert sp(lat.BLUME_CAPEL, 0.0, b) == 1
    assert sp(lat.BLUME_CAPEL, 0.0, 0.3) == 0 and sp(lat.BLUME_CAPEL, 0.0, 0.0) == 0
    assert sp(lat.BLUME_CAPEL, 0.7, workloads.BETA_BC) == 0
    L = 1024
    g = lat.Lattice(L, lat.BLUME_CAPEL, 0.0, 70707, scheme)
    o = oracle.OracleLattice(L, lat.BLUME_CAPEL, 0.0, 70707, scheme)
    sched = [specials[0], specials[0], 0.3, specials[3], specials[4], 0.0, specials[1], 0.55, specials[2], specials[4]]
    for b in sched:                                   # one sweep per call: two plain launches each
        g.sweep([b])
    o.sweep(sched)
    assert g.specialised_launches == 2 * sum(1 for b in sched if b in specials)
    assert np.array_equal(g.get_spins(), o.get_spins())
    for fill in (1, 0, -1):                           # ordered states: every lane deciding, ties most frequent
        g.fill(fill)
        o.set_spins(np.full((L, L), fill, dtype=np.int8))
        for b in (specials[0], specials[3], specials[4]):
            g.sweep([b]); o.sweep([b])
        assert np.array_equal(g.get_spins(), o.get_spins()), fill
    _same_measure(g, o, 48, L, 0.0)
    g.close(); o.close()


def test_plane_case_specialised_kernels_are_bit_identical():
    """Launch-time specialisation (compile-time LOP3 truth tables for the betas the workloads run at):
    the specialised instantiations run -- the launch-kind counter says so -- and give the oracle's
    trajectory; a beta without an instantiation takes the generic brx.idx kernel in between."""
    L = 4608                                          # large enough for the marching kernel (not one row per thread)
    specials = [BETA_C, 1.0 / 1.66, 1.0 / 2.27414861561203, BETA_C / 1.01]
    for b in specials:
        assert lat.lib().lattice_plane_case_specialised(lat.ISING, 0.0, b) == 1
    assert lat.lib().lattice_plane_case_specialised(lat.ISING, 0.0, 0.3) == 0
    assert lat.lib().lattice_plane_case_specialised(lat.ISING, 0.0, 0.35) == 0
    assert lat.lib().lattice_plane_case_specialised(lat.ISING, 0.0, 0.0) == 0
    g = lat.Lattice(L, lat.ISING, 0.0, 60606)
    o = oracle.OracleLattice(L, lat.ISING, 0.0, 60606)
    sched = [BETA_C, BETA_C, 0.3, 1.0 / 1.66, 1.0 / 1.66, 0.0, 1.0 / 2.27414861561203, BETA_C / 1.01, 0.35, BETA_C]
    for b in sched:                                   # one sweep per call: two plain launches each
        g.sweep([b])
    o.sweep(sched)
    assert g.specialised_launches == 2 * sum(1 for b in sched if b in specials)
    assert np.array_equal(g.get_spins(), o.get_spins())
    # from the all-up state: every lane needs a decision, ties are most frequent
    g.fill(1)
    o.set_spins(np.ones((L, L), dtype=np.int8))
    for b in (BETA_C, 1.0 / 1.66, 1.0 / 2.27414861561203):
        g.sweep([b]); o.sweep([b])
    assert np.array_equal(g.get_spins(), o.get_spins())
    g.close(); o.close()
    # the batched marching kernel has the same instantiations
    seeds = np.array([1, 2, 3, 4], dtype=np.uint64)
    bt = lat.LatticeBatch(L, seeds)
    for b in (BETA_C, 0.3, BETA_C / 1.01):
        bt.sweep([b])
    for k in (0, 3):
        o = oracle.OracleLattice(L, lat.ISING, 0.0, int(seeds[k]))
        o.sweep([BETA_C, 0.3, BETA_C / 1.01])
        assert np.array_equal(bt.get_spins(k), o.get_spins())
        o.close()
    assert int(lat.lib().lattice_specialised_launches(bt._h)) == 4
    bt.close()


def test_ising_infinite_temperature_flips_every_spin():
    g = lat.Lattice(512, lat.ISING, 0.0, 3)
    s0 = g.get_spins()
    M0, Q0, Sx0, Sy0 = g.measure(16)
    g.sweep([0.0])
    assert np.array_equal(g.get_spins(), -s0)
    M1, Q1, Sx1, Sy1 = g.measure(16)
    assert M1 == -M0 and np.array_equal(Sx0, Sx1) and np.array_equal(Sy0, Sy1)


def test_zero_temperature_fixed_point_and_single_defect():
    L = 256
    g = lat.Lattice(L, lat.ISING, 0.0, 3)
    up = np.ones((L, L), dtype=np.int8)
    g.set_spins(up)
    g.sweep([math.inf] * 3)
    assert np.array_equal(g.get_spins(), up)
    d = up.copy()
    d[17, 33] = -1
    d[200, 0] = -1
    g.set_spins(d)
    g.sweep([math.inf])
    assert np.array_equal(g.get_spins(), up)
    M, Q, Sx, Sy = g.measure(L // 2)
    assert M == L * L and (Sx == L * L).all() and (Sy == L * L).all()


@pytest.mark.parametrize("name", ["ising_L2p16_ramp", "bc_L2p15_ramp"])
def test_protocol2_schedule_small(name):
    """BASELINE.json config 5's beta(t) ramp on a small lattice: thresholds change every sweep."""
    w = workloads.CONFIGS[name]
    L = 256
    g = lat.Lattice(L, w.model, w.delta, w.seed)
    o = oracle.OracleLattice(L, w.model, w.delta, w.seed)
    sched = w.beta_schedule(1100)
    assert len(np.unique(sched)) == 1000
    beta = sched[::11]                       # 100 distinct values spanning the ramp and the plateau
    g.sweep(beta)
    o.sweep(beta)
    assert np.array_equal(g.get_spins(), o.get_spins())
    _same_measure(g, o, 64, L, w.delta)


@pytest.mark.parametrize("name", ["ising_L2p16_twostep", "bc_L2p16_twostep"])
def test_paper_two_step_schedule_small(name):
    """The paper's protocol 2 (Table II): T_1 until t_switch, then T_2 -- on a
    small lattice, across the switch (set_time moves both sides next to t_switch)."""
    w = workloads.CONFIGS[name]
    L = 256
    g = lat.Lattice(L, w.model, w.delta, w.seed)
    o = oracle.OracleLattice(L, w.model, w.delta, w.seed)
    t0 = w.t_switch - 12
    sched = w.beta_schedule(30, t0)
    assert sched[11] == w.beta_1 and sched[12] == w.beta_f and len(np.unique(sched)) == 2
    g.sweep(w.beta_schedule(10))
    o.sweep(w.beta_schedule(10))
    g.set_time(t0)
    o.close()
    o = oracle.OracleLattice.window(L, w.model, w.delta, w.seed, 1, t0, 0, 0, g.get_spins())
    g.sweep(sched)
    o.sweep(sched)
    assert g.time == o.time == t0 + 30
    assert np.array_equal(g.get_spins(), o.get_spins())


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
def test_special_states_and_set_get_roundtrip(model):
    L = 128
    g = lat.Lattice(L, model, 0.0, 9)
    o = oracle.OracleLattice(L, model, 0.0, 9)
    rng = np.random.default_rng(1)
    vals = np.array([-1, 1] if model == lat.ISING else [-1, 0, 1], dtype=np.int8)
    i, j = np.indices((L, L))
    for s in (np.ones((L, L), np.int8), np.where((i + j) % 2 == 0, 1, -1).astype(np.int8),
              np.where(i % 2 == 0, 1, -1).astype(np.int8), np.where(j % 4 < 2, 1, -1).astype(np.int8),
              rng.choice(vals, (L, L))):
        g.set_spins(s)
        o.set_spins(s)
        assert np.array_equal(g.get_spins(), s)
        _same_measure(g, o, L // 2, L)
    # windows with periodic wrap
    win = rng.choice(vals, (40, 70))
    g.set_spins(win, 100, 90)
    o.set_spins(win, 100, 90)
    assert np.array_equal(g.get_spins(), o.get_spins())
    assert np.array_equal(g.get_spins(100, 90, 40, 70), win)
    if model == lat.ISING:
        with pytest.raises(lat.LatticeError):
            g.set_spins(np.zeros((2, 2), np.int8))


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
def test_measure_rows_partition(model):
    L = 256
    g = lat.Lattice(L, model, 0.0, 21)
    o = oracle.OracleLattice(L, model, 0.0, 21)
    beta = BETA_C if model == lat.ISING else workloads.BETA_BC
    g.sweep([beta] * 20)
    o.sweep([beta] * 20)
    tot = None
    for i0, n in ((0, 1), (1, 100), (101, 155)):
        _same_measure(g, o, 100, L, rows=(i0, n))
        M, Q, Sx, Sy = g.measure(100, (i0, n))
        part = np.concatenate([[M, Q], Sx, Sy])
        tot = part if tot is None else tot + part
    M, Q, Sx, Sy = g.measure(100)
    assert np.array_equal(tot, np.concatenate([[M, Q], Sx, Sy]))


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
@pytest.mark.parametrize("L,r_max", [(1024, 512), (1536, 100), (2048, 131)])
def test_measure_blocked_kernels_all_r_and_ragged_slabs(L, r_max, model):
    """The row-blocked measurement kernels (16-row blocks, 16-word segments, chunks of 64 r):
    every r up to L/2 on the whole lattice, and slabs whose row count is not a multiple of 16."""
    g = lat.Lattice(L, model, 0.0, 1234 + L)
    o = oracle.OracleLattice(L, model, 0.0, 1234 + L)
    beta = BETA_C if model == lat.ISING else workloads.BETA_BC
    g.sweep([beta] * 30)
    o.sweep([beta] * 30)
    _same_measure(g, o, r_max, L)
    for i0, n in ((0, 16), (3, 45), (L - 33, 33), (500, 7)):
        _same_measure(g, o, min(r_max, 70), L, rows=(i0, n))


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
@pytest.mark.parametrize("L", [64, 192, 1024, 1536, 2048])
def test_measure_list_sparse_r(L, model):
    """lattice_measure_list (the paper's sparse sampling in r): every listed r equals
    the oracle's dense count at that r -- log-spaced lists, unsorted lists with repeats, r = 1 and
    r = L/2, whole lattice and ragged row ranges (list kernels + generic remainder)."""
    g = lat.Lattice(L, model, 0.0, 4321 + L)
    o = oracle.OracleLattice(L, model, 0.0, 4321 + L)
    beta = BETA_C if model == lat.ISING else workloads.BETA_BC
    g.sweep([beta] * 12)
    o.sweep([beta] * 12)
    half = L // 2
    Mo, Qo, Sxo, Syo = o.measure(half)
    lists = [sorted({max(1, int(round(half ** (k / 40)))) for k in range(41)}),
             [half, 1, 2, 1, half - 1, 33, 33, 17][: 8 if half > 33 else 5],
             [3], list(range(1, min(half, 70) + 1))]
    for rl in lists:
        rl = [r for r in rl if 1 <= r <= half]
        M, Q, Sx, Sy = g.measure_list(rl)
        assert (M, Q) == (Mo, Qo)
        assert Sx.tolist() == [int(Sxo[r - 1]) for r in rl], rl
        assert Sy.tolist() == [int(Syo[r - 1]) for r in rl], rl
    for i0, n in ((0, 16), (3, 45), (L - 33, 33), (L // 2, 7), (1, 1)):
        rl = [1, 2, 5, half // 2, half]
        Ms, Qs, Sxs, Sys = o.measure(half, (i0, n))
        M, Q, Sx, Sy = g.measure_list(rl, (i0, n))
        assert (M, Q) == (Ms, Qs)
        assert Sx.tolist() == [int(Sxs[r - 1]) for r in rl] and Sy.tolist() == [int(Sys[r - 1]) for r in rl]
    with pytest.raises(lat.LatticeError):
        g.measure_list([0])
    with pytest.raises(lat.LatticeError):
        g.measure_list([half + 1])
    g.close(); o.close()


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
@pytest.mark.parametrize("L", [256, 768, 2048])
def test_measure_r1_single_pass(L, model):
    """r_max = 1 (the per-step record e, m, q) goes through the one-pass marching kernel."""
    g = lat.Lattice(L, model, 0.4, 99 + L)
    o = oracle.OracleLattice(L, model, 0.4, 99 + L)
    _same_measure(g, o, 1, L, 0.4)
    beta = BETA_C if model == lat.ISING else workloads.BETA_BC
    g.sweep([beta] * 10)
    o.sweep([beta] * 10)
    _same_measure(g, o, 1, L, 0.4)
    for i0, n in ((0, 1), (1, 1), (0, 32), (5, 64), (L - 71, 71), (31, 2), (L - 1, 1)):
        _same_measure(g, o, 1, L, rows=(i0, n))


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
def test_fill_ordered_states_and_sweep_from_them(model):
    """lattice_fill: ordered states (bench.py's worst-case input), then sweeps against the oracle."""
    L = 512
    g = lat.Lattice(L, model, 0.0, 77)
    o = oracle.OracleLattice(L, model, 0.0, 77)
    for spin in ([1, -1] if model == lat.ISING else [1, 0, -1]):
        g.fill(spin)
        want = np.full((L, L), spin, dtype=np.int8)
        assert np.array_equal(g.get_spins(), want)
        M, Q, Sx, Sy = g.measure(8)
        assert M == spin * L * L and Q == abs(spin) * L * L and (Sx == Q).all() and (Sy == Q).all()
        o.set_spins(want)
        beta = [BETA_C if model == lat.ISING else workloads.BETA_BC] * 6
        g.sweep(beta)
        o.sweep(beta)
        assert np.array_equal(g.get_spins(), o.get_spins()), spin
    if model == lat.ISING:
        with pytest.raises(lat.LatticeError):
            g.fill(0)
    with pytest.raises(lat.LatticeError):
        g.fill(2)


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
@pytest.mark.parametrize("L", [256, 512, 1024])
def test_scheme2_64_bit_thresholds(L, model):
    """RNG scheme 2 (56-bit tails, 64-bit thresholds) against the oracle's scheme 2, including
    temperatures so low that the 32-bit table has only zeros where the 64-bit one does not."""
    g = lat.Lattice(L, model, 0.0, 2024 + L, scheme=2)
    o = oracle.OracleLattice(L, model, 0.0, 2024 + L, scheme=2)
    bc = BETA_C if model == lat.ISING else workloads.BETA_BC
    beta = [bc] * 8 + [3.0, 3.0, 0.0, 0.05, 25.0, math.inf] + [bc / 1.01] * 8
    g.sweep(beta[:5])                       # several calls: launch path and persistent path
    g.sweep(beta[5:6])
    g.sweep(beta[6:])
    o.sweep(beta)
    assert np.array_equal(g.get_spins(), o.get_spins())
    _same_measure(g, o, 32, L)
    # scheme 2 differs from scheme 1 only on a 2^-32 tie: same trajectory here
    g1 = lat.Lattice(L, model, 0.0, 2024 + L, scheme=1)
    g1.sweep(beta)
    assert np.array_equal(g.get_spins(), g1.get_spins())
    g.close(); g1.close(); o.close()


def test_scheme2_needs_marching_kernels():
    with pytest.raises(lat.LatticeError):
        lat.Lattice(64, lat.ISING, 0.0, 1, scheme=2)                 # L not a multiple of 256
    b = lat.Lattice(256, lat.BLUME_CAPEL, 5.5, 1, scheme=2)          # |Delta| > 4: only the generic kernel
    with pytest.raises(lat.LatticeError):
        b.sweep([0.5])
    b.close()


@pytest.mark.parametrize("scheme", [1, 2])
@pytest.mark.parametrize("L,delta,T", [(256, 0.7, 1.2), (512, -1.3, 2.0), (1024, 1.965, 0.6), (2048, 1.965, 0.9),
                                       (256, 3.5, 1.0), (512, -4.0, 1.5), (256, 4.0, 0.8), (768, -0.25, 1.7)])
def test_blume_capel_marching_kernel_with_crystal_field(L, delta, T, scheme):
    """Delta != 0 on the marching path (bc_march_row_gen): vacate and occupy have their own
    thresholds and x <= 0 is not "always" for them (Eq. 1).  Spins and counts
    against the oracle, including sweeps at beta = 0, at very low temperature and from ordered
    states (every lane deciding, ties most frequent)."""
    g = lat.Lattice(L, lat.BLUME_CAPEL, delta, 8800 + L, scheme)
    o = oracle.OracleLattice(L, lat.BLUME_CAPEL, delta, 8800 + L, scheme)
    sched = [1.0 / T] * 8 + [0.0, 0.05, 4.0, math.inf, 1.0 / T]
    n0 = g.launches
    g.sweep(sched[:3])
    g.sweep(sched[3:])
    assert g.launches - n0 == 2 * len(sched)
    o.sweep(sched)
    assert np.array_equal(g.get_spins(), o.get_spins())
    _same_measure(g, o, min(L // 2, 48), L, delta)
    for spin in (1, 0, -1):
        g.fill(spin)
        o.set_spins(np.full((L, L), spin, dtype=np.int8))
        g.sweep([1.0 / T] * 3)
        o.sweep([1.0 / T] * 3)
        assert np.array_equal(g.get_spins(), o.get_spins()), spin
    g.close(); o.close()


def test_randomised_parity_sweep_of_parameters():
    """Seeded random (model, L, scheme, beta schedule, Delta, seed) cases: spins and counts after a
    few sweeps, bit for bit.  Covers the generic kernels (L not a multiple of 256, scheme 0,
    Delta != 0) next to the marching ones, and per-sweep threshold changes."""
    rng = np.random.default_rng(20250314)
    for case in range(24):
        model = int(rng.integers(0, 2))
        L = int(rng.choice([64, 128, 192, 256, 320, 512, 768]))
        scheme = int(rng.integers(0, 2))
        delta = float(rng.choice([0.0, 0.0, rng.uniform(-2, 2)])) if model == lat.BLUME_CAPEL else 0.0
        seed = int(rng.integers(0, 2 ** 63))
        n = int(rng.integers(3, 9))
        beta = rng.uniform(0.0, 1.2, size=n)
        if case % 5 == 0:
            beta[int(rng.integers(0, n))] = 0.0                 # an "always accept" sweep in the middle
        g = lat.Lattice(L, model, delta, seed, scheme)
        o = oracle.OracleLattice(L, model, delta, seed, scheme)
        g.sweep(beta)
        o.sweep(beta)
        assert np.array_equal(g.get_spins(), o.get_spins()), (case, model, L, scheme, delta, seed)
        _same_measure(g, o, int(rng.integers(1, L // 2 + 1)), L, delta)
        g.close(); o.close()


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
def test_determinism_and_checkpoint_resume(model):
    L = 512
    beta = [0.4] * 10
    a = lat.Lattice(L, model, 0.2, 8)
    a.sweep(beta + beta)
    b = lat.Lattice(L, model, 0.2, 8)
    b.sweep(beta)
    snap, t = b.get_spins(), b.time
    c = lat.Lattice(L, model, 0.2, 999)          # different start, then restored
    c2 = lat.Lattice(L, model, 0.2, 8)
    c2.set_spins(snap)
    c2.set_time(t)
    c2.sweep(beta)
    assert np.array_equal(a.get_spins(), c2.get_spins())
    assert not np.array_equal(a.get_spins(), c.get_spins())
    a.close(); b.close(); c.close(); c2.close()


def test_api_errors_on_device():
    g = lat.Lattice(64, lat.ISING, 0.0, 1)
    with pytest.raises(lat.LatticeError):
        g.sweep([-0.1])
    with pytest.raises(lat.LatticeError):
        g.sweep([math.nan])
    with pytest.raises(lat.LatticeError):
        g.measure(33)
    with pytest.raises(lat.LatticeError):
        g.measure(0)
    g.sweep([0.3])
    with pytest.raises(lat.LatticeError) as e:
        lat.binding.Lattice._check(g, lat.lib().lattice_set_rng_scheme(g._h, 0), "set_rng_scheme")
    assert e.value.status == lat.binding.ESTATE
    assert g.launches == 3                         # init + two half-sweeps
    # a view is a measurement-only handle: windows, set_time and set_rng_scheme are refused
    import ctypes as C
    import torch
    rows = 96
    buf = torch.zeros(2 * rows * (256 // 64) * 4, dtype=torch.uint8, device="cuda")
    h = C.c_void_p()
    L_ = lat.lib()
    assert L_.lattice_view(C.byref(h), 256, lat.ISING, rows, C.c_void_p(buf.data_ptr()), buf.numel(), None) == 0
    out = np.zeros((4, 4), dtype=np.int8)
    p8 = out.ctypes.data_as(C.POINTER(C.c_int8))
    assert L_.lattice_get_spins(h, 0, 0, 4, 4, p8) == lat.binding.ESTATE
    assert L_.lattice_get_spins(h, 200, 0, 4, 4, p8) == lat.binding.ESTATE      # i >= rows: was out of bounds
    assert L_.lattice_set_spins(h, 0, 0, 4, 4, p8) == lat.binding.ESTATE
    assert L_.lattice_set_time(h, 5) == lat.binding.ESTATE
    assert L_.lattice_set_rng_scheme(h, 0) == lat.binding.ESTATE
    assert L_.lattice_fill(h, 1) == lat.binding.EINVAL
    L_.lattice_destroy(h)


def test_first_half_sweep_acceptance_closed_form():
    """No oracle: on an i.i.d. start the first black half-sweep at beta_c flips a fraction
    11/16 + (sqrt2-1)^2/4 + (sqrt2-1)^4/16 of the black spins (SURVEY 8c pins)."""
    L = 4096
    g = lat.Lattice(L, lat.ISING, 0.0, 12345)
    s0 = g.get_spins()
    g.half_sweep(0, BETA_C)
    s1 = g.get_spins()
    i, j = np.indices((L, L))
    black = (i + j) % 2 == 0
    assert np.array_equal(s0[~black], s1[~black])
    frac = float((s0[black] != s1[black]).mean())
    a = math.sqrt(2) - 1
    want = 11 / 16 + a ** 2 / 4 + a ** 4 / 16
    sigma = math.sqrt(want * (1 - want) / black.sum())
    assert abs(frac - want) < 5 * sigma
