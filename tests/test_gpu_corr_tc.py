"""Dense C(r) on the tensor cores (csrc/corr_tc.cuh, lattice_set_measure_path(2)) against the oracle's
literal double loops and against the XOR/popcount kernels: the same exact integers for both models,
both axes, several passes of 512 partner positions, periodic wrap, ragged row ranges and ordered
states (where every product has the same sign and the accumulators reach their largest values)."""
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


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
@pytest.mark.parametrize("L,r_max", [(1024, 512), (1024, 60), (2048, 700), (1536, 768)])
def test_tensor_core_correlations_equal_oracle_and_popcount_path(L, r_max, model):
    g = lat.Lattice(L, model, 0.0, 31415 + L)
    o = oracle.OracleLattice(L, model, 0.0, 31415 + L)
    beta = workloads.BETA_C_ISING if model == lat.ISING else workloads.BETA_BC
    g.sweep([beta] * 20)
    o.sweep([beta] * 20)
    want = o.measure(r_max)
    g.set_measure_path(1)
    pop = g.measure(r_max)
    g.set_measure_path(2)
    tc = g.measure(r_max)
    g.set_measure_path(3)                           # CTA pairs (tcgen05 cta_group::2, csrc/corr_tc2.cuh) on both axes
    tc2 = g.measure(r_max)
    g.set_measure_path(4)                           # one CTA per item (csrc/corr_tc.cuh) on both axes
    tc1 = g.measure(r_max)
    for got in (pop, tc, tc2, tc1):
        assert (got[0], got[1]) == (want[0], want[1])
        assert np.array_equal(got[2], want[2]), np.nonzero(got[2] != want[2])[0][:8]
        assert np.array_equal(got[3], want[3]), np.nonzero(got[3] != want[3])[0][:8]
    # row ranges: partner rows wrap periodically, base rows end inside a 128-row tile
    for i0, n in ((0, 128), (5, 300), (L - 77, 77), (L // 2 - 1, 1)):
        ws = o.measure(min(r_max, 200), (i0, n))
        for path in (2, 3, 4):
            g.set_measure_path(path)
            gs = g.measure(min(r_max, 200), (i0, n))
            assert (gs[0], gs[1]) == (ws[0], ws[1]) and np.array_equal(gs[2], ws[2]) and np.array_equal(gs[3], ws[3]), (i0, n, path)
    # ordered and striped states: |G| = L, every accumulator at its extreme
    i, j = np.indices((L, L))
    for s in (np.ones((L, L), np.int8), np.where(i % 2 == 0, 1, -1).astype(np.int8),
              np.where(j % 4 < 2, 1, -1).astype(np.int8)):
        g.set_spins(s)
        o.set_spins(s)
        b = o.measure(r_max)
        for path in (2, 3, 4):
            g.set_measure_path(path)
            a = g.measure(r_max)
            assert (a[0], a[1]) == (b[0], b[1]) and np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3]), path
    g.close(); o.close()


def test_transposed_bands_with_a_row_length_that_is_not_a_power_of_two():
    """L = 6144 = 3 * 2048: 96 words per row, 24 pair tiles, the partner windows wrap at a tile boundary."""
    L, r_max = 6144, 600
    g = lat.Lattice(L, lat.ISING, 0.0, 14142)
    o = oracle.OracleLattice(L, lat.ISING, 0.0, 14142)
    g.sweep([workloads.BETA_C_ISING] * 5)
    o.sweep([workloads.BETA_C_ISING] * 5)
    for path in (2, 3, 4):
        g.set_measure_path(path)
        for rows in (None, (2048, 3072)):
            a, b = g.measure(r_max, rows), o.measure(r_max, rows)
            assert (a[0], a[1]) == (b[0], b[1]) and np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3]), (path, rows)
    g.close(); o.close()


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
def test_x_axis_on_the_transposed_bands(model):
    """L a multiple of 2048: the x axis of the tensor-core path runs the y-axis pair kernel on a
    transposed copy of whole 512-row bands (csrc/corr_transpose.cuh) and the MN-major kernel on the
    rows that are left; odd first rows and short ranges take the MN-major kernel alone.  All of it
    against the oracle."""
    L, r_max = 4096, 300
    g = lat.Lattice(L, model, 0.0, 27182)
    o = oracle.OracleLattice(L, model, 0.0, 27182)
    beta = workloads.BETA_C_ISING if model == lat.ISING else workloads.BETA_BC
    g.sweep([beta] * 8)
    o.sweep([beta] * 8)
    g.set_measure_path(2)
    for rows in (None, (0, 1536), (1024, 700), (1, 600), (2048, 2048), (3584, 512)):
        n0 = g.launches
        a, b = g.measure(r_max, rows), o.measure(r_max, rows)
        assert (a[0], a[1]) == (b[0], b[1]) and np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3]), rows
        if rows in (None, (2048, 2048), (3584, 512)):
            assert g.launches - n0 == 1 + 1 + 2           # M/Q, y axis, transpose + x axis on the copy
    g.close(); o.close()


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
def test_tensor_core_path_on_a_view(model):
    """A measurement-only view (not periodic along y; how a slab measures C(r) for r > 1): base rows
    0..1023 of a buffer holding rows 0..1023+r_max of an L = 4096 lattice take the tensor-core path by
    themselves (x axis on the transposed band) and give the oracle's partial sums."""
    L, n, r_max = 4096, 1024, 300
    g = lat.Lattice(L, model, 0.0, 16180)
    o = oracle.OracleLattice(L, model, 0.0, 16180)
    beta = workloads.BETA_C_ISING if model == lat.ISING else workloads.BETA_BC
    g.sweep([beta] * 6)
    o.sweep([beta] * 6)
    planes = 2 if model == lat.ISING else 4
    rows = n + r_max
    import torch
    g.synchronize()
    view = g.buf.view(planes, L, L // 64 * 4)[:, :rows].contiguous()
    torch.cuda.synchronize()
    M, Q, Sx, Sy = lat.binding.measure_buffer(L, model, rows, n, r_max, view.data_ptr(), view.numel(),
                                                 g.stream.cuda_stream)
    Mo, Qo, Sxo, Syo = o.measure(r_max, (0, n))
    assert (M, Q) == (Mo, Qo) and np.array_equal(Sx, Sxo) and np.array_equal(Sy, Syo)
    g.close(); o.close()


def test_tensor_core_path_selection_and_errors():
    g = lat.Lattice(256, lat.ISING, 0.0, 1)
    with pytest.raises(lat.LatticeError):
        g.set_measure_path(2)                       # L < 1024
    with pytest.raises(lat.LatticeError):
        g.set_measure_path(3)                       # CTA pairs: the same shape conditions
    with pytest.raises(lat.LatticeError):
        g.set_measure_path(5)
    g.set_measure_path(1)
    g.close()
    b = lat.LatticeBatch(1024, np.arange(3, dtype=np.uint64) + 5)
    b.sweep([workloads.BETA_C_ISING] * 6)
    import ctypes as C
    assert lat.lib().lattice_set_measure_path(b._h, 2) == 0
    M, Q, Sx, Sy = b.measure(130)
    for k in range(3):
        o = oracle.OracleLattice(1024, lat.ISING, 0.0, 5 + k)
        o.sweep([workloads.BETA_C_ISING] * 6)
        Mo, Qo, Sxo, Syo = o.measure(130)
        assert (M[k], Q[k]) == (Mo, Qo) and np.array_equal(Sx[k], Sxo) and np.array_equal(Sy[k], Syo)
        o.close()
    b.close()
