"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

A whole-lattice oracle is out of reach at L = 2^15 .. 2^20 (up to 7e13 updates), so parity is
checked on sampled outputs the oracle can compute one by one:

* windowed replay -- download an (h+4s) x (w+4s) window, run s sweeps on the GPU, download the
  inner h x w block; the oracle evolves the window with global (i, j) keying and frozen garbage
  outside.  The dependency cone grows 2 sites per sweep, so the inner block must match bit for
  bit.  Windows are placed on the periodic wrap, on the row-slab boundaries of the marching
  kernels (multiples of 32 rows), on 128-bit run boundaries (multiples of 256 columns) and at
  seeded random positions.
* slab measurements -- `lattice_measure_rows` on a few rows against the oracle's per-spin pair
  sums on the downloaded rows for r in {1, 2, 31, 32, 33, ..., r_max-1, r_max}; and the slab
  sums of a partition of the rows add up to the whole-lattice counts.
"""
import os

import numpy as np
import pytest

import oracle
import paper_2503_14688_b200 as lat
from paper_2503_14688_b200 import workloads

pytestmark = pytest.mark.gpu
NCPU = os.cpu_count() or 1


@pytest.fixture(autouse=True)
def _threads():
    oracle.set_threads(NCPU)
    yield
    oracle.set_threads(1)


def _fits(w):
    import torch
    free, _ = torch.cuda.mem_get_info(0)
    return free > w.state_bytes + (3 << 30)


def _windows(L, rng, h, w):
    """(i0, j0) origins of the inner blocks: wrap corner, slab/run boundaries, random."""
    fixed = [(L - h // 2, L - w // 2),                 # wraps both axes
             (32 * (L // 64) - 7, 256 * (L // 512) - 9),  # crosses a 32-row slab and a 128-bit run
             (0, 0), (L // 2 - 3, L - w + 5)]
    rnd = [(int(rng.integers(0, L)), int(rng.integers(0, L))) for _ in range(4)]
    return [(i % L, j % L) for i, j in fixed + rnd]


def _replay(g, w, t_start, s, h=40, wd=300):
    """Windowed replay of sweeps t_start .. t_start+s-1 (g must be at time t_start)."""
    L, m = w.L, 2 * s
    rng = np.random.default_rng(w.seed)
    wins = _windows(L, rng, h, wd)
    before = [g.get_spins((i0 - m) % L, (j0 - m) % L, h + 2 * m, wd + 2 * m) for i0, j0 in wins]
    beta = w.beta_schedule(s, t_start)
    assert g.time == t_start
    g.sweep(beta)
    for (i0, j0), b in zip(wins, before):
        outside = 1 if w.model == lat.ISING else 0
        o = oracle.OracleLattice.window(L, w.model, w.delta, w.seed, 1, t_start, (i0 - m) % L,
                                        (j0 - m) % L, b, outside=outside)
        o.sweep(beta)
        want = o.get_spins(m, m, h, wd)
        got = g.get_spins(i0, j0, h, wd)
        assert np.array_equal(got, want), (w.name, t_start, i0, j0)
        # the test bites: the window did change
        assert not np.array_equal(got, b[m:m + h, m:m + wd])
        o.close()


def _slab_counts(g, w, i0, n, rs):
    """Oracle per-spin sums over base rows i0..i0+n-1 from downloaded rows."""
    L = w.L
    base = g.get_spins(i0, 0, n, L)
    ones = np.ones(L, dtype=np.int8)
    M = sum(oracle.pair_sum(base[a], ones) for a in range(n))
    Q = sum(oracle.pair_sum(base[a], base[a]) for a in range(n))
    Sx, Sy = {}, {}
    for r in rs:
        Sx[r] = sum(oracle.pair_sum(base[a], base[a], r) for a in range(n))
        part = g.get_spins((i0 + r) % L, 0, n, L)
        Sy[r] = sum(oracle.pair_sum(base[a], part[a]) for a in range(n))
    return M, Q, Sx, Sy


def _check_slab(g, w, i0, n, r_max):
    rs = sorted({r for r in (1, 2, 3, 31, 32, 33, 63, 64, 65, 127, 128, 129, 1023, 1024, 1025,
                             r_max - 1, r_max) if 1 <= r <= r_max})
    M, Q, Sx, Sy = g.measure(r_max, (i0, n))
    Mo, Qo, Sxo, Syo = _slab_counts(g, w, i0, n, rs)
    assert (M, Q) == (Mo, Qo)
    M1, Q1, Sx1, Sy1 = g.measure(1, (i0, n))                 # the one-pass r_max = 1 kernel
    assert (M1, Q1, Sx1[0], Sy1[0]) == (Mo, Qo, Sxo[1], Syo[1])
    for r in rs:
        assert Sx[r - 1] == Sxo[r], ("Sx", r)
        assert Sy[r - 1] == Syo[r], ("Sy", r)
    # the sparse-list call on the same slab: the same separations, handed over unsorted
    rl = rs[::-1]
    Ml, Ql, Sxl, Syl = g.measure_list(rl, (i0, n))
    assert (Ml, Ql) == (Mo, Qo)
    assert Sxl.tolist() == [Sxo[r] for r in rl] and Syl.tolist() == [Syo[r] for r in rl]


@pytest.mark.parametrize("name,t_late,r_slab", [("ising_L2p20", 0, 4096), ("ising_L2p16_ramp", 990, 1024),
                                                ("bc_L2p15_ramp", 990, 1024), ("bc_L16384", 64, 4096),
                                                ("ising_L4096", 1000, 1024)])
def test_full_size_windowed_replay_and_slab_measurements(name, t_late, r_slab):
    w = workloads.CONFIGS[name]
    if not _fits(w):
        pytest.skip(f"{name}: {w.state_bytes >> 30} GiB does not fit on this device")
    g = lat.Lattice(w.L, w.model, w.delta, w.seed)
    L = w.L
    # the disordered start itself, on sampled windows
    rng = np.random.default_rng(1)
    for i0, j0 in _windows(L, rng, 16, 300):
        got = g.get_spins(i0, j0, 16, 300)
        o = oracle.lib().oracle_initial_spin
        rows = [(i0 + a) % L for a in (0, 7, 15)]
        for a, i in zip((0, 7, 15), rows):
            want = [o(w.seed, w.model, L, i, (j0 + b) % L) for b in range(300)]
            assert got[a].tolist() == want
    _replay(g, w, 0, 3)                          # sweeps 0..2 from the disordered start
    if t_late > g.time:                          # later in the run (domains have formed; for the
        g.sweep(w.beta_schedule(t_late - g.time, g.time))   # ramp: the thresholds change per sweep)
    _replay(g, w, g.time, 3)
    if name == "ising_L2p20":                    # constant beta_c: the plane-case specialised kernel ran
        assert g.specialised_launches == 2 * 6
    # a sweep counter with the high bit set keys correctly too
    g.set_time(3_000_000_000)
    _replay(g, w, 3_000_000_000, 2)
    # measurements: slabs against the oracle, partition against the whole
    _check_slab(g, w, 5, 3, min(r_slab, L // 2))
    _check_slab(g, w, L - 2, 2, min(r_slab, L // 2))          # partner rows wrap around
    r_small = 2
    whole = g.measure(r_small)
    cuts = [0, 37, L // 2 + 16, L]
    tot = None
    for a, b in zip(cuts[:-1], cuts[1:]):
        M, Q, Sx, Sy = g.measure(r_small, (a, b - a))
        part = np.concatenate([[M, Q], Sx, Sy])
        tot = part if tot is None else tot + part
    assert np.array_equal(tot, np.concatenate([[whole[0], whole[1]], whole[2], whole[3]]))
    one = g.measure(1)
    assert (one[0], one[1], one[2][0], one[3][0]) == (whole[0], whole[1], whole[2][0], whole[3][0])
    if w.model == lat.ISING:
        assert whole[1] == L * L
    g.close()


def test_config2_ising_L4096_first_sweeps_whole_lattice():
    """BASELINE.json config 2 from the start, whole lattice against the oracle, records at 2^k."""
    w = workloads.CONFIGS["ising_L4096"]
    g = lat.Lattice(w.L, w.model, w.delta, w.seed)
    o = oracle.OracleLattice(w.L, w.model, w.delta, w.seed)
    done = 0
    for t in w.measure_times(64):
        if t > done:
            beta = w.beta_schedule(t - done, done)
            g.sweep(beta)
            o.sweep(beta)
            done = t
        assert np.array_equal(g.get_spins(), o.get_spins()), t
        r_max = 64 if t < 64 else w.r_max
        Mg, Qg, Sxg, Syg = g.measure(r_max)
        Mo, Qo, Sxo, Syo = o.measure(r_max)
        assert (Mg, Qg) == (Mo, Qo) and np.array_equal(Sxg, Sxo) and np.array_equal(Syg, Syo)
        xg, rg = lat.xi(Sxg, Syg, Qg, w.L)
        xo, ro = oracle.xi(Sxo, Syo, Qo, w.L)
        assert rg == ro and (xg == xo or abs(xg - xo) <= 1e-12 * abs(xo))
    g.close()


def test_config3_blume_capel_L16384_first_sweeps_whole_lattice():
    """BASELINE.json config 3 from the start: 4 sweeps of the whole 2^28-site lattice."""
    w = workloads.CONFIGS["bc_L16384"]
    g = lat.Lattice(w.L, w.model, w.delta, w.seed)
    o = oracle.OracleLattice(w.L, w.model, w.delta, w.seed)
    beta = w.beta_schedule(4)
    g.set_persist_blocks(1 << 20)                 # bc_persist_kernel on request: one cooperative launch
    n0 = g.launches
    g.sweep(beta[:2])
    assert g.launches - n0 == 1
    g.set_persist_blocks(0)                       # the default at this size: two launches per sweep
    g.sweep(beta[2:])
    assert g.launches - n0 == 5
    o.sweep(beta)
    for i0 in (0, 8191, 16384 - 512):            # compare in row bands to bound host memory
        assert np.array_equal(g.get_spins(i0, 0, 512, w.L), o.get_spins(i0, 0, 512, w.L))
    Mg, Qg, Sxg, Syg = g.measure(8)
    Mo, Qo, Sxo, Syo = o.measure(8)
    assert (Mg, Qg) == (Mo, Qo) and np.array_equal(Sxg, Sxo) and np.array_equal(Syg, Syo)
    g.close()
