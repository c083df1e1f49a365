"""GPU parity of batched replicas (lattice_create_batch): every replica of a batch must be bit for
bit the stand-alone lattice with its seed, i.e. equal to the oracle run with that seed -- spins and
integer counts -- whichever kernel the batch takes: the register-resident tiny kernel (L = 64, 128,
all sweeps in one launch), the batched marching kernel (L a multiple of 256, replica = blockIdx.y),
or the per-replica fall-back (other L, scheme 0, Blume-Capel)."""
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


def _check_replicas(b, model, delta, scheme, sched, which, r_max):
    M, Q, Sx, Sy = b.measure(r_max)
    for k in which:
        o = oracle.OracleLattice(b.L, model, delta, int(b.seeds[k]), scheme)
        o.sweep(sched)
        assert np.array_equal(b.get_spins(k), o.get_spins()), (b.L, k)
        Mo, Qo, Sxo, Syo = o.measure(r_max)
        assert (M[k], Q[k]) == (Mo, Qo), k
        assert np.array_equal(Sx[k], Sxo) and np.array_equal(Sy[k], Syo), k
        M1, Q1, Sx1, Sy1 = b.measure_replica(k, r_max)
        assert (M1, Q1) == (Mo, Qo) and np.array_equal(Sx1, Sxo) and np.array_equal(Sy1, Syo)
        o.close()


@pytest.mark.parametrize("L,n_rep,scheme", [(64, 1, 1), (64, 37, 1), (128, 5, 1), (128, 64, 2), (64, 600, 1)])
def test_tiny_replicas_all_sweeps_in_one_launch(L, n_rep, scheme):
    if scheme == 2:
        pytest.skip("scheme 2 needs L % 256 == 0")
    seeds = 777000 + 13 * np.arange(n_rep, dtype=np.uint64)
    b = lat.LatticeBatch(L, seeds, lat.ISING, 0.0, scheme)
    sched = [BETA_C] * 20 + [0.0, 0.3, math.inf, 1e-9] + [BETA_C / 1.01] * 17
    n0 = b.launches
    b.sweep(sched[:1])
    b.sweep(sched[1:])
    assert b.launches - n0 == 2                       # one launch per call, however many sweeps
    assert b.time == len(sched)
    which = sorted({0, n_rep - 1, n_rep // 2, min(n_rep - 1, 16), min(n_rep - 1, 17)})
    _check_replicas(b, lat.ISING, 0.0, scheme, sched, which, L // 2)
    b.close()


@pytest.mark.parametrize("L", [64, 128])
def test_single_small_lattice_takes_the_register_resident_kernel(L):
    """A plain (non-batch) Ising lattice with L = 64 / 128: lattice_sweep(n >= 2) is one launch of
    ising_tiny_kernel with one replica, equal to the oracle and to one sweep per call."""
    g = lat.Lattice(L, lat.ISING, 0.0, 4711 + L)
    s = lat.Lattice(L, lat.ISING, 0.0, 4711 + L)
    o = oracle.OracleLattice(L, lat.ISING, 0.0, 4711 + L)
    for sched in ([BETA_C] * 40, [BETA_C, 0.0, 0.3, math.inf, 1e-9, BETA_C / 1.01] * 3):
        n0 = g.launches
        g.sweep(sched)
        assert g.launches - n0 == 1
        n0 = s.launches
        for b in sched:
            s.sweep([b])
        assert s.launches - n0 == 2 * len(sched)
        o.sweep(sched)
        assert np.array_equal(g.get_spins(), o.get_spins())
        assert np.array_equal(s.get_spins(), o.get_spins())
    assert g.time == s.time == o.time
    Mg, Qg, Sxg, Syg = g.measure(L // 2)
    Mo, Qo, Sxo, Syo = o.measure(L // 2)
    assert (Mg, Qg) == (Mo, Qo) and np.array_equal(Sxg, Sxo) and np.array_equal(Syg, Syo)
    g.close(); s.close(); o.close()


def test_config1_as_a_batch_is_one_launch_and_equals_the_single_lattice():
    """BASELINE config 1 (L = 64, 2000 sweeps at beta_c): replica 0 carries the config's own seed."""
    w = workloads.CONFIGS["ising_L64"]
    seeds = np.array([w.seed + 1000 * k for k in range(64)], dtype=np.uint64)
    b = lat.LatticeBatch(w.L, seeds, w.model, w.delta)
    g = lat.Lattice(w.L, w.model, w.delta, w.seed)
    o = oracle.OracleLattice(w.L, w.model, w.delta, w.seed)
    done = 0
    for t in w.measure_times():
        if t > done:
            beta = w.beta_schedule(t - done, done)
            n0 = b.launches
            b.sweep(beta)
            assert b.launches - n0 == 1
            g.sweep(beta)
            o.sweep(beta)
            done = t
        want = o.get_spins()
        assert np.array_equal(b.get_spins(0), want), t
        assert np.array_equal(g.get_spins(), want), t
        M, Q, Sx, Sy = b.measure(w.r_max)
        Mo, Qo, Sxo, Syo = o.measure(w.r_max)
        assert (M[0], Q[0]) == (Mo, Qo) and np.array_equal(Sx[0], Sxo) and np.array_equal(Sy[0], Syo)
    b.close(); g.close(); o.close()


@pytest.mark.parametrize("L,n_rep,scheme,one_by_one", [(256, 7, 1, True), (512, 3, 1, True), (1024, 130, 1, True),
                                                       (2048, 2, 2, False), (4096, 3, 1, False)])
def test_marching_batch_replica_in_grid_y(L, n_rep, scheme, one_by_one):
    """ising_march_batch_kernel: L >= 768, or any L % 256 == 0 when sweeps are issued one per call."""
    seeds = 424200 + 101 * np.arange(n_rep, dtype=np.uint64)
    b = lat.LatticeBatch(L, seeds, lat.ISING, 0.0, scheme)
    sched = [BETA_C] * 4 + [0.0, 0.6] + [BETA_C / 1.01] * 3
    n0 = b.launches
    if one_by_one:
        for beta in sched:
            b.sweep([beta])
    else:
        b.sweep(sched)
    chunks = (n_rep + 127) // 128
    assert b.launches - n0 == 2 * len(sched) * chunks        # two launches per sweep per chunk of 128
    which = sorted({0, n_rep - 1, n_rep // 2, min(n_rep - 1, 128)})
    _check_replicas(b, lat.ISING, 0.0, scheme, sched, which, min(L // 2, 40))
    b.close()


@pytest.mark.parametrize("L,n_rep,scheme", [(256, 7, 1), (256, 300, 2), (512, 33, 1), (768, 5, 1), (1024, 40, 1)])
def test_block_per_replica_kernel_all_sweeps_in_one_launch(L, n_rep, scheme):
    """ising_block_kernel (256 <= L <= 512, n >= 2): one block per replica, block barriers between colours.
    From L = 768 on two launches of the batched marching kernel per sweep are measured faster and taken."""
    seeds = 909000 + 7 * np.arange(n_rep, dtype=np.uint64)
    b = lat.LatticeBatch(L, seeds, lat.ISING, 0.0, scheme)
    sched = [BETA_C] * 7 + [0.0, 0.6, math.inf] + [BETA_C / 1.01] * 6
    n0 = b.launches
    b.sweep(sched[:9])
    b.sweep(sched[9:])
    assert b.launches - n0 == (2 if L <= 512 else 2 * len(sched) * ((n_rep + 127) // 128))
    which = sorted({0, n_rep - 1, n_rep // 2})
    _check_replicas(b, lat.ISING, 0.0, scheme, sched, which, min(L // 2, 40))
    b.close()


@pytest.mark.parametrize("model,L,delta,scheme", [(lat.ISING, 192, 0.0, 1), (lat.ISING, 256, 0.0, 0),
                                                  (lat.BLUME_CAPEL, 256, 0.0, 1), (lat.BLUME_CAPEL, 128, 0.7, 0)])
def test_fallback_one_launch_per_replica(model, L, delta, scheme):
    seeds = np.array([5, 6, 2 ** 63 + 11], dtype=np.uint64)
    b = lat.LatticeBatch(L, seeds, model, delta, scheme)
    beta = BETA_C if model == lat.ISING else workloads.BETA_BC
    sched = [beta] * 5 + [0.2]
    b.sweep(sched)
    _check_replicas(b, model, delta, scheme, sched, [0, 1, 2], L // 2)
    b.close()


def test_batch_handle_api_rules():
    seeds = np.arange(4, dtype=np.uint64)
    b = lat.LatticeBatch(256, seeds)
    L_ = lat.lib()
    import ctypes as C
    assert L_.lattice_replicas(b._h) == 4
    out = np.zeros((4, 4), dtype=np.int8)
    p8 = out.ctypes.data_as(C.POINTER(C.c_int8))
    assert L_.lattice_get_spins(b._h, 0, 0, 4, 4, p8) == lat.binding.ESTATE          # per-lattice call on the batch
    kid = b._replica(2)
    beta = np.array([0.4])
    assert L_.lattice_sweep(kid, 1, beta.ctypes.data_as(C.POINTER(C.c_double))) == lat.binding.ESTATE
    assert L_.lattice_set_time(kid, 3) == lat.binding.ESTATE
    assert L_.lattice_destroy(kid) == lat.binding.ESTATE
    h = C.c_void_p()
    assert L_.lattice_replica(b._h, 4, C.byref(h)) == lat.binding.EINVAL
    # fill and set_spins through a replica, then the batch measures it
    b.fill(1)
    s = -np.ones((2, 256), dtype=np.int8)
    b.set_spins(1, s, 10, 0)
    M, Q, Sx, Sy = b.measure(2)
    assert M.tolist() == [256 * 256, 256 * 256 - 4 * 256, 256 * 256, 256 * 256]
    # checkpoint-style restore: set_time on the batch, sweeps continue from there for all replicas
    b.set_time(1000)
    b.sweep([0.5])
    assert b.time == 1001
    b.close()
