"""ctypes loader for the CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package (see oracle/oracle.h).  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")

ISING, BLUME_CAPEL = 0, 1
OK, EINVAL, ENOMEM, ESTATE = 0, -1, -2, -4


def build(force: bool = False) -> str:
    """Compile oracle.c -> liboracle.so with gcc (plain C11, -O2, OpenMP over rows)."""
    src = os.path.join(_HERE, "oracle.c")
    hdr = os.path.join(_HERE, "oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    import fcntl
    with open(_SO + ".lock", "w") as lock:           # several ranks may build at once
        fcntl.flock(lock, fcntl.LOCK_EX)
        if (not force and os.path.exists(_SO)
                and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
            return _SO
        tmp = f"{_SO}.{os.getpid()}.tmp"
        cmd = ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-fopenmp", "-shared", "-fPIC",
               src, "-o", tmp, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _SO)
    return _SO


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(build())
    u32p, u64p, i64p, i8p, f64p = (C.POINTER(C.c_uint32), C.POINTER(C.c_uint64),
                                   C.POINTER(C.c_int64), C.POINTER(C.c_int8),
                                   C.POINTER(C.c_double))
    vp = C.c_void_p
    sig = {
        "oracle_philox4x32_10": (None, [u32p, u32p, u32p]),
        "oracle_u32": (C.c_uint32, [C.c_uint64, C.c_int, C.c_uint32, C.c_int, C.c_uint64]),
        "oracle_u64": (C.c_uint64, [C.c_uint64, C.c_uint32, C.c_int, C.c_uint64]),
        "oracle_thresholds64": (None, [C.c_int, C.c_double, C.c_double, u64p, C.POINTER(C.c_ubyte)]),
        "oracle_proposal_bit": (C.c_int, [C.c_uint64, C.c_uint32, C.c_int, C.c_uint64]),
        "oracle_initial_spin": (C.c_int, [C.c_uint64, C.c_int, C.c_uint32, C.c_uint64, C.c_uint64]),
        "oracle_thresholds": (None, [C.c_int, C.c_double, C.c_double, u64p]),
        "oracle_create": (C.c_int, [C.POINTER(vp), C.c_uint32, C.c_int, C.c_double, C.c_uint64]),
        "oracle_window_create": (C.c_int, [C.POINTER(vp), C.c_uint32, C.c_int, C.c_double,
                                           C.c_uint64, C.c_int, C.c_uint64, C.c_uint64,
                                           C.c_uint64, C.c_uint32, C.c_uint32, i8p, C.c_int]),
        "oracle_set_rng_scheme": (C.c_int, [vp, C.c_int]),
        "oracle_sweep": (C.c_int, [vp, C.c_uint64, f64p]),
        "oracle_half_sweep": (C.c_int, [vp, C.c_int, C.c_double]),
        "oracle_measure": (C.c_int, [vp, C.c_uint32, i64p, i64p, i64p, i64p]),
        "oracle_measure_rows": (C.c_int, [vp, C.c_uint64, C.c_uint64, C.c_uint32, i64p, i64p,
                                          i64p, i64p]),
        "oracle_get_spins": (C.c_int, [vp, C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, i8p]),
        "oracle_set_spins": (C.c_int, [vp, C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, i8p]),
        "oracle_run_series": (C.c_int, [vp, C.c_uint64, C.c_double, i64p, i64p, i64p, i64p]),
        "oracle_pair_sum": (C.c_int64, [i8p, i8p, C.c_uint64, C.c_uint64]),
        "oracle_time": (C.c_uint64, [vp]),
        "oracle_xi": (C.c_double, [i64p, i64p, C.c_uint32, C.c_int64, C.c_uint32, u32p]),
        "oracle_energy": (C.c_double, [i64p, i64p, C.c_int64, C.c_double, C.c_uint32]),
        "oracle_destroy": (C.c_int, [vp]),
        "oracle_set_threads": (None, [C.c_int]),
        "oracle_get_threads": (C.c_int, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


def _p(a: np.ndarray, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def u32(seed, scheme, t, colour, P) -> int:
    return int(lib().oracle_u32(seed, scheme, t, colour, P))


def u64(seed, t, colour, P) -> int:
    return int(lib().oracle_u64(seed, t, colour, P))


def thresholds64(model, delta, beta):
    """(thr[n] on the 2^64 scale, always[n]) for scheme 2."""
    n = 2 if model == ISING else 54
    thr = np.zeros(n, dtype=np.uint64)
    alw = np.zeros(n, dtype=np.uint8)
    lib().oracle_thresholds64(model, float(delta), float(beta), _p(thr, C.c_uint64), _p(alw, C.c_ubyte))
    return thr, alw


def proposal_bit(seed, t, colour, P) -> int:
    return int(lib().oracle_proposal_bit(seed, t, colour, P))


def thresholds(model, delta, beta) -> np.ndarray:
    out = np.zeros(2 if model == ISING else 54, dtype=np.uint64)
    lib().oracle_thresholds(model, float(delta), float(beta), _p(out, C.c_uint64))
    return out


def pair_sum(a: np.ndarray, b: np.ndarray, shift: int = 0) -> int:
    a = np.ascontiguousarray(a, dtype=np.int8)
    b = np.ascontiguousarray(b, dtype=np.int8)
    assert a.size == b.size
    return int(lib().oracle_pair_sum(_p(a, C.c_int8), _p(b, C.c_int8), a.size, shift))


def xi(Sx, Sy, Q, L):
    Sx = np.ascontiguousarray(Sx, dtype=np.int64)
    Sy = np.ascontiguousarray(Sy, dtype=np.int64)
    rc = C.c_uint32(0)
    v = lib().oracle_xi(_p(Sx, C.c_int64), _p(Sy, C.c_int64), Sx.size, int(Q), int(L), C.byref(rc))
    return float(v), int(rc.value)


def energy(Sx, Sy, Q, delta, L) -> float:
    Sx = np.ascontiguousarray(Sx, dtype=np.int64)
    Sy = np.ascontiguousarray(Sy, dtype=np.int64)
    return float(lib().oracle_energy(_p(Sx, C.c_int64), _p(Sy, C.c_int64), int(Q), float(delta),
                                     int(L)))


def set_threads(n: int) -> None:
    lib().oracle_set_threads(int(n))


def get_threads() -> int:
    return int(lib().oracle_get_threads())


class OracleError(RuntimeError):
    pass


def _check(rc: int, what: str) -> None:
    if rc != OK:
        raise OracleError(f"{what} failed with status {rc}")


class OracleLattice:
    """Thin handle around oracle_lattice_t (host memory, one int8 per site)."""

    def __init__(self, L, model=ISING, delta=0.0, seed=0, scheme=1, _handle=None, _shape=None):
        self.L, self.model, self.delta, self.seed = int(L), int(model), float(delta), int(seed)
        if _handle is not None:
            self._h, self.shape = _handle, _shape
            return
        h = C.c_void_p()
        _check(lib().oracle_create(C.byref(h), self.L, self.model, self.delta, self.seed),
               "oracle_create")
        self._h, self.shape = h, (self.L, self.L)
        _check(lib().oracle_set_rng_scheme(self._h, int(scheme)), "oracle_set_rng_scheme")

    @classmethod
    def window(cls, Lg, model, delta, seed, scheme, t0, i0, j0, spins, outside=1):
        spins = np.ascontiguousarray(spins, dtype=np.int8)
        hh, ww = spins.shape
        h = C.c_void_p()
        _check(lib().oracle_window_create(C.byref(h), int(Lg), int(model), float(delta), int(seed),
                                          int(scheme), int(t0), int(i0), int(j0), hh, ww,
                                          _p(spins, C.c_int8), int(outside)),
               "oracle_window_create")
        return cls(Lg, model, delta, seed, _handle=h, _shape=(hh, ww))

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    __del__ = close

    @property
    def time(self) -> int:
        return int(lib().oracle_time(self._h))

    def sweep(self, beta) -> None:
        b = np.ascontiguousarray(np.atleast_1d(beta), dtype=np.float64)
        _check(lib().oracle_sweep(self._h, b.size, _p(b, C.c_double)), "oracle_sweep")

    def half_sweep(self, colour: int, beta: float) -> None:
        _check(lib().oracle_half_sweep(self._h, int(colour), float(beta)), "oracle_half_sweep")

    def measure(self, r_max: int, rows=None):
        Sx = np.zeros(r_max, dtype=np.int64)
        Sy = np.zeros(r_max, dtype=np.int64)
        M, Q = C.c_int64(0), C.c_int64(0)
        if rows is None:
            rc = lib().oracle_measure(self._h, r_max, C.byref(M), C.byref(Q), _p(Sx, C.c_int64),
                                      _p(Sy, C.c_int64))
        else:
            rc = lib().oracle_measure_rows(self._h, rows[0], rows[1], r_max, C.byref(M),
                                           C.byref(Q), _p(Sx, C.c_int64), _p(Sy, C.c_int64))
        _check(rc, "oracle_measure")
        return int(M.value), int(Q.value), Sx, Sy

    def run_series(self, n: int, beta: float, with_state: bool = False):
        M = np.zeros(n, dtype=np.int64)
        B = np.zeros(n, dtype=np.int64)
        Q = np.zeros(n, dtype=np.int64)
        S = np.zeros(n, dtype=np.int64) if with_state else None
        _check(lib().oracle_run_series(self._h, n, float(beta), _p(M, C.c_int64),
                                       _p(B, C.c_int64), _p(Q, C.c_int64),
                                       _p(S, C.c_int64) if with_state else None),
               "oracle_run_series")
        return M, B, Q, S

    def get_spins(self, i0=0, j0=0, h=None, w=None) -> np.ndarray:
        h = self.shape[0] if h is None else h
        w = self.shape[1] if w is None else w
        out = np.zeros((h, w), dtype=np.int8)
        _check(lib().oracle_get_spins(self._h, i0, j0, h, w, _p(out, C.c_int8)), "oracle_get_spins")
        return out

    def set_spins(self, spins, i0=0, j0=0) -> None:
        s = np.ascontiguousarray(spins, dtype=np.int8)
        _check(lib().oracle_set_spins(self._h, i0, j0, s.shape[0], s.shape[1], _p(s, C.c_int8)),
               "oracle_set_spins")
