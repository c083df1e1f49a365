"""lattice_measure_static: the measurement entry point that allocates nothing (counters in a file-scope
device array, include/lattice.h).  Its counts must equal lattice_measure's -- exact integers, the same
bar as every other GPU test -- on two calls in a row (the second call finds the first call's counts in
the shared array and has to clear them), alone in a fresh process or after the other tests.

This file is named so that pytest collects it last: the suite runs with `pytest -x`."""
import numpy as np
import pytest

import paper_2503_14688_b200 as lat
from paper_2503_14688_b200 import binding, workloads

pytestmark = pytest.mark.gpu


def _same(a, b):
    return a[0] == b[0] and a[1] == b[1] and np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3])


@pytest.mark.parametrize("model,L,r_max", [(lat.ISING, 1024, 256), (lat.BLUME_CAPEL, 1024, 100), (lat.ISING, 2048, 1024),
                                           (lat.ISING, 192, 96)])
def test_static_measure_equals_the_allocating_path_on_two_calls_in_a_row(model, L, r_max):
    beta = workloads.BETA_C_ISING if model == lat.ISING else workloads.BETA_BC
    g = lat.Lattice(L, model, 0.0, 31337 + L)
    g.set_measure_path(1)                       # the allocating path on the same XOR/popcount kernels
    g.sweep([beta] * 5)
    want1 = g.measure(r_max)
    got1 = g.measure_static(r_max)              # first call
    assert _same(got1, want1)
    g.sweep([beta] * 3)                         # another state: other counts in every entry
    got2 = g.measure_static(r_max)              # second call right after the first: stale counts cleared
    want2 = g.measure(r_max)
    assert _same(got2, want2)
    assert not np.array_equal(got1[2], got2[2])
    # a shorter range after a longer one, and r_max = 1 (the one-pass kernel), on the same shared array
    assert _same(g.measure_static(7), g.measure(7))
    assert _same(g.measure_static(1), g.measure(1))
    # default measurement path (tensor cores where they apply) gives the same counts too
    g.set_measure_path(0)
    assert _same(g.measure_static(r_max), g.measure(r_max))
    g.close()


def test_static_measure_rejects_sizes_beyond_the_maximum():
    g = lat.Lattice(4096, lat.ISING, 0.0, 5)
    assert binding.STATIC_RMAX == 1024
    with pytest.raises(lat.LatticeError) as e:
        g.measure_static(binding.STATIC_RMAX + 1)            # <= L/2, but beyond the static array
    assert e.value.status == binding.EINVAL and "LATTICE_STATIC_RMAX" in str(e.value)
    with pytest.raises(lat.LatticeError):
        g.measure_static(0)
    assert _same(g.measure_static(binding.STATIC_RMAX), g.measure(binding.STATIC_RMAX))
    g.close()
    b = lat.LatticeBatch(256, np.arange(2, dtype=np.uint64))
    import ctypes as C
    M, Q = C.c_int64(0), C.c_int64(0)
    S = (C.c_int64 * 4)()
    assert lat.lib().lattice_measure_static(b._h, 1, C.byref(M), C.byref(Q), S, S) == binding.ESTATE
    b.close()
