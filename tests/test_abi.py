"""CPU-only checks of the C-ABI boundary: the library loads, exports every symbol that
include/lattice.h declares, and its host-only helpers (thresholds, xi, energy, argument
validation) agree with the oracle.  No device work is started here."""
import ctypes as C
import math
import os
import re

import numpy as np
import pytest

import oracle
import paper_2503_14688_b200 as lat
from paper_2503_14688_b200 import binding, workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "lattice.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lattice_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    L = lat.lib()
    declared = _declared_symbols()
    assert len(declared) >= 18
    for name in declared:
        assert hasattr(L, name), name
    assert sorted(binding.SIGNATURES) == declared        # the binding covers the whole header


def test_state_bytes():
    assert lat.state_bytes(64, lat.ISING) == 512
    assert lat.state_bytes(4096, lat.ISING) == 2 << 20
    assert lat.state_bytes(1 << 20, lat.ISING) == 128 << 30
    assert lat.state_bytes(16384, lat.BLUME_CAPEL) == 64 << 20
    for bad in (0, 32, 65, 100, (1 << 20) + 64):
        assert lat.state_bytes(bad, lat.ISING) == 0
    assert lat.state_bytes(64, 7) == 0


def test_thresholds_equal_oracle_on_every_config_schedule():
    for w in workloads.CONFIGS.values():
        betas = np.unique(w.beta_schedule(min(w.sweeps, 1200)))
        for beta in betas:
            assert np.array_equal(lat.thresholds(w.model, w.delta, beta),
                                  oracle.thresholds(w.model, w.delta, beta)), (w.name, beta)


@pytest.mark.parametrize("delta", [0.0, 0.7, -1.3, 2.0, -50.0])
def test_thresholds_equal_oracle_general(delta):
    for beta in (0.0, 1e-9, 0.1, 0.44068679350977147, 1 / 1.6934, 1.0, 3.0, 25.0, math.inf):
        for model in (lat.ISING, lat.BLUME_CAPEL):
            a, b = lat.thresholds(model, delta, beta), oracle.thresholds(model, delta, beta)
            assert np.array_equal(a, b)
            assert a.max() <= 1 << 32


def test_blume_capel_table_has_the_mirror_symmetry_the_kernel_uses():
    # the kernel indexes thresholds by (move type, x); entries related by s -> -s, h -> -h
    # must therefore be identical in the 54-entry table
    for delta in (0.0, 0.7, -1.3):
        t = lat.thresholds(lat.BLUME_CAPEL, delta, 0.61).reshape(3, 2, 9)
        for h in range(-4, 5):
            assert t[2, 0, h + 4] == t[0, 1, -h + 4]       # flip
            assert t[2, 1, h + 4] == t[0, 0, -h + 4]       # vacate
            assert t[1, 0, h + 4] == t[1, 1, -h + 4]       # occupy


def test_xi_and_energy_equal_oracle():
    rng = np.random.default_rng(5)
    for _ in range(50):
        r_max = int(rng.integers(1, 200))
        Sx = rng.integers(-1000, 100000, r_max)
        Sy = rng.integers(-1000, 100000, r_max)
        a, ra = lat.xi(Sx, Sy, 4096, 64)
        b, rb = oracle.xi(Sx, Sy, 4096, 64)
        assert ra == rb and (a == b or abs(a - b) <= 1e-12 * abs(b))
        assert lat.energy(Sx, Sy, 4000, 0.3, 64) == oracle.energy(Sx, Sy, 4000, 0.3, 64)


def test_xi_closed_form():
    # S(r) ~ x^r with x = exp(-1/a): untruncated sums give coth(1/2a) (SURVEY 8c pins)
    for a, want in ((5.0, 10.0333111), (50.0, 100.003333311)):
        r = np.arange(1, 6001)
        S = np.round(1e17 * np.exp(-r / a)).astype(np.int64)
        S = S[S > 0]
        v, rc = lat.xi(S, S, 1, 1 << 20)
        assert abs(v - 1.0 / math.tanh(1 / (2 * a))) < 2e-6 * want


def test_create_rejects_bad_arguments_before_touching_the_device():
    L = lat.lib()
    h = C.c_void_p()
    fake = C.c_void_p(0x1000)      # never dereferenced: validation fails first
    assert L.lattice_create(C.byref(h), 65, 0, 0.0, 1, fake, 1 << 20, None) == binding.EINVAL
    assert L.lattice_create(C.byref(h), 64, 5, 0.0, 1, fake, 1 << 20, None) == binding.EINVAL
    assert L.lattice_create(C.byref(h), 64, 0, math.nan, 1, fake, 1 << 20, None) == binding.EINVAL
    assert L.lattice_create(C.byref(h), 64, 0, 0.0, 1, fake, 511, None) == binding.EINVAL
    assert L.lattice_create(C.byref(h), 64, 0, 0.0, 1, C.c_void_p(0x1004), 512, None) == binding.EINVAL
    assert L.lattice_create(C.byref(h), 64, 0, 0.0, 1, None, 512, None) == binding.EINVAL
    assert L.lattice_create(None, 64, 0, 0.0, 1, fake, 512, None) == binding.EINVAL
    assert L.lattice_sweep(None, 1, None) == binding.EINVAL
    assert L.lattice_destroy(None) == binding.EINVAL
    assert L.lattice_strerror(binding.ECUDA) == b"CUDA error"


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError, match="no CPU path"):
        lat.Lattice(64)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2503_14688_b200")
    pat = re.compile(r"^\s*(import|from)\s+oracle\b|liboracle|oracle\.h|oracle/", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dirpath, f)).read()), f


def test_slab_bytes_and_create_slab_argument_checks():
    """Row-slab mode (include/lattice.h): sizes and the checks made before touching a device."""
    import ctypes as C
    L = lat.lib()
    wpr = 1024 // 64
    assert L.lattice_slab_bytes(1024, lat.ISING, 256) == 2 * (256 + 2) * wpr * 4
    assert L.lattice_slab_bytes(1024, lat.ISING, 1024) == 2 * (1024 + 2) * wpr * 4
    assert L.lattice_slab_bytes(1024, lat.BLUME_CAPEL, 256) == 4 * (256 + 2) * wpr * 4
    for bad in [(1000, lat.ISING, 64), (64, lat.ISING, 64), (1024, lat.ISING, 100), (1024, lat.ISING, 0),
                (1024, lat.ISING, 2048), (1024, 7, 256)]:
        assert L.lattice_slab_bytes(*bad) == 0, bad
    h = C.c_void_p()
    fake = C.c_void_p(0x10000)
    n = L.lattice_slab_bytes(1024, lat.ISING, 256)
    for args in [(1024, lat.ISING, 0.0, 1, 32, 256, fake, n, None),        # row0 not a multiple of 64
                 (1024, lat.ISING, 0.0, 1, 896, 256, fake, n, None),       # runs past the last row
                 (1024, lat.ISING, 0.0, 1, 0, 256, fake, n - 1, None),     # buffer too small
                 (1024, lat.ISING, 0.0, 1, 0, 256, None, n, None),         # no buffer
                 (1024, lat.ISING, float("nan"), 1, 0, 256, fake, n, None)]:
        assert L.lattice_create_slab(C.byref(h), *args) == lat.binding.EINVAL, args
    assert L.lattice_slab_set_neighbours(None, fake, 64, fake, 64) == lat.binding.EINVAL


def test_view_and_copy_argument_checks():
    import ctypes as C
    L = lat.lib()
    h = C.c_void_p()
    fake = C.c_void_p(0x10000)
    need = 2 * 300 * (1024 // 64) * 4
    assert L.lattice_view(C.byref(h), 1024, lat.ISING, 300, fake, need - 1, None) == lat.binding.EINVAL
    assert L.lattice_view(C.byref(h), 1000, lat.ISING, 300, fake, need, None) == lat.binding.EINVAL
    assert L.lattice_view(C.byref(h), 1024, lat.ISING, 0, fake, need, None) == lat.binding.EINVAL
    assert L.lattice_view(C.byref(h), 1024, lat.ISING, 300, None, need, None) == lat.binding.EINVAL
    assert L.lattice_view(C.byref(h), 1024, lat.ISING, 300, fake, need, None) == lat.binding.OK
    M, Q = C.c_int64(), C.c_int64()
    S = (C.c_int64 * 64)()
    # base rows + r_max must fit in the view (it is not periodic along y); checked before any launch
    assert L.lattice_measure_rows(h, 0, 280, 40, C.byref(M), C.byref(Q), S, S) == lat.binding.EINVAL
    assert L.lattice_half_sweep(h, 0, 0.4) == lat.binding.ESTATE          # a view cannot be swept
    assert L.lattice_destroy(h) == lat.binding.OK
    assert L.lattice_device_copy(None, fake, 16, None) == lat.binding.EINVAL
    assert L.lattice_device_copy(fake, fake, 0, None) == lat.binding.OK


@pytest.mark.parametrize("model,delta", [(lat.ISING, 0.0), (lat.BLUME_CAPEL, 0.0), (lat.BLUME_CAPEL, -1.3),
                                         (lat.BLUME_CAPEL, 0.7)])
def test_thresholds64_equal_oracle(model, delta):
    """RNG scheme 2: the library's 64-bit thresholds equal the oracle's, entry by entry."""
    import math
    for beta in (0.0, 1e-12, 0.2, workloads.BETA_C_ISING, workloads.BETA_BC, 1.0, 3.0, 11.0, 50.0, math.inf):
        tg, ag = lat.thresholds64(model, delta, beta)
        to, ao = oracle.thresholds64(model, delta, beta)
        assert np.array_equal(tg, to) and np.array_equal(ag, ao), beta


def test_plane_case_specialisations_match_the_config_betas():
    """The hard-coded plane-case constants of ising_march.cuh are the ones the thresholds of the
    workloads' betas give (host-only: the library derives the cases from lattice_thresholds)."""
    f = lat.lib().lattice_plane_case_specialised
    for name in ("ising_L64", "ising_L4096", "ising_L2p20"):
        w = workloads.CONFIGS[name]
        assert f(w.model, w.delta, float(w.beta_schedule(1)[0])) == 1, name
    w = workloads.CONFIGS["ising_L2p16_twostep"]
    assert f(w.model, 0.0, w.beta_1) == 1 and f(w.model, 0.0, w.beta_f) == 1
    w = workloads.CONFIGS["ising_L2p16_ramp"]
    assert f(w.model, 0.0, w.beta_f) == 1                       # the plateau after the ramp
    assert f(lat.ISING, 0.0, 0.2) == 0
    # Blume-Capel: the truth-table sets of bc_march.cuh (config 3, the paper's T_c, both two-step temperatures,
    # the plateau of config 5b's ramp); no set for another beta or for a crystal field
    for name in ("bc_L16384", "bc_L2p19", "bc_L2p15_ramp"):
        w = workloads.CONFIGS[name]
        assert f(w.model, w.delta, w.beta_f) == 1, name
    w = workloads.CONFIGS["bc_L2p16_twostep"]
    assert f(w.model, 0.0, w.beta_1) == 1 and f(w.model, 0.0, w.beta_f) == 1
    assert f(lat.BLUME_CAPEL, 0.0, 0.3) == 0 and f(lat.BLUME_CAPEL, 0.7, workloads.BETA_BC) == 0
