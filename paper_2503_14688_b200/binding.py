"""Thin ctypes binding of include/lattice.h: argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used for the
device buffer and the stream, nothing else.  There is no CPU fallback: if the shared library is
missing or no CUDA device is present, constructing a `Lattice` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import buildlib as _build

ISING, BLUME_CAPEL = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, -1, -2, -3, -4

_lib = None

_u32p, _u64p, _i64p, _i8p, _f64p = (C.POINTER(C.c_uint32), C.POINTER(C.c_uint64),
                                    C.POINTER(C.c_int64), C.POINTER(C.c_int8),
                                    C.POINTER(C.c_double))
_vp = C.c_void_p

#: name -> (restype, argtypes); one entry per symbol declared in include/lattice.h
SIGNATURES = {
    "lattice_state_bytes": (C.c_size_t, [C.c_uint32, C.c_int]),
    "lattice_create": (C.c_int, [C.POINTER(_vp), C.c_uint32, C.c_int, C.c_double, C.c_uint64,
                                 _vp, C.c_size_t, _vp]),
    "lattice_batch_bytes": (C.c_size_t, [C.c_uint32, C.c_uint32, C.c_int]),
    "lattice_create_batch": (C.c_int, [C.POINTER(_vp), C.c_uint32, C.c_uint32, C.c_int, C.c_double, _u64p,
                                       _vp, C.c_size_t, _vp]),
    "lattice_replicas": (C.c_uint32, [_vp]),
    "lattice_replica": (C.c_int, [_vp, C.c_uint32, C.POINTER(_vp)]),
    "lattice_measure_batch": (C.c_int, [_vp, C.c_uint32, _i64p, _i64p, _i64p, _i64p]),
    "lattice_slab_bytes": (C.c_size_t, [C.c_uint32, C.c_int, C.c_uint32]),
    "lattice_create_slab": (C.c_int, [C.POINTER(_vp), C.c_uint32, C.c_int, C.c_double, C.c_uint64,
                                      C.c_uint32, C.c_uint32, _vp, C.c_size_t, _vp]),
    "lattice_slab_set_flags": (C.c_int, [_vp, _vp, _vp, _vp]),
    "lattice_slab_set_neighbours": (C.c_int, [_vp, _vp, C.c_uint32, _vp, C.c_uint32]),
    "lattice_view": (C.c_int, [C.POINTER(_vp), C.c_uint32, C.c_int, C.c_uint32, _vp, C.c_size_t, _vp]),
    "lattice_device_copy": (C.c_int, [_vp, _vp, C.c_size_t, _vp]),
    "lattice_enable_peer_access": (C.c_int, [C.c_int, C.c_int]),
    "lattice_device_alloc": (C.c_int, [C.POINTER(_vp), C.c_size_t]),
    "lattice_device_free": (C.c_int, [_vp]),
    "lattice_ipc_export": (C.c_int, [_vp, C.POINTER(C.c_ubyte)]),
    "lattice_ipc_open": (C.c_int, [C.POINTER(C.c_ubyte), C.POINTER(_vp)]),
    "lattice_ipc_close": (C.c_int, [_vp]),
    "lattice_set_rng_scheme": (C.c_int, [_vp, C.c_int]),
    "lattice_sweep": (C.c_int, [_vp, C.c_uint64, _f64p]),
    "lattice_sweep_record": (C.c_int, [_vp, C.c_uint64, _f64p, _i64p, _i64p, _i64p, _i64p]),
    "lattice_half_sweep": (C.c_int, [_vp, C.c_int, C.c_double]),
    "lattice_measure": (C.c_int, [_vp, C.c_uint32, _i64p, _i64p, _i64p, _i64p]),
    "lattice_measure_static": (C.c_int, [_vp, C.c_uint32, _i64p, _i64p, _i64p, _i64p]),
    "lattice_measure_rows": (C.c_int, [_vp, C.c_uint64, C.c_uint64, C.c_uint32, _i64p, _i64p,
                                       _i64p, _i64p]),
    "lattice_measure_list": (C.c_int, [_vp, C.c_uint64, C.c_uint64, _u32p, C.c_uint32, _i64p, _i64p, _i64p, _i64p]),
    "lattice_get_spins": (C.c_int, [_vp, C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, _i8p]),
    "lattice_set_spins": (C.c_int, [_vp, C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, _i8p]),
    "lattice_fill": (C.c_int, [_vp, C.c_int]),
    "lattice_time": (C.c_uint64, [_vp]),
    "lattice_set_time": (C.c_int, [_vp, C.c_uint64]),
    "lattice_launches": (C.c_uint64, [_vp]),
    "lattice_set_persist_blocks": (C.c_int, [_vp, C.c_uint32]),
    "lattice_set_measure_path": (C.c_int, [_vp, C.c_int]),
    "lattice_specialised_launches": (C.c_uint64, [_vp]),
    "lattice_plane_case_specialised": (C.c_int, [C.c_int, C.c_double, C.c_double]),
    "lattice_thresholds": (None, [C.c_int, C.c_double, C.c_double, _u64p]),
    "lattice_thresholds64": (None, [C.c_int, C.c_double, C.c_double, _u64p, C.POINTER(C.c_ubyte)]),
    "lattice_xi": (C.c_double, [_i64p, _i64p, C.c_uint32, C.c_int64, C.c_uint32, _u32p]),
    "lattice_energy": (C.c_double, [_i64p, _i64p, C.c_int64, C.c_double, C.c_uint32]),
    "lattice_ubench_int_dispatch": (C.c_int, [C.c_int, _vp, _f64p, _f64p]),
    "lattice_destroy": (C.c_int, [_vp]),
    "lattice_strerror": (C.c_char_p, [C.c_int]),
    "lattice_last_error": (C.c_char_p, [_vp]),
}


def lib() -> C.CDLL:
    """Load liblattice.so (building it with nvcc if the sources are newer)."""
    global _lib
    if _lib is not None:
        return _lib
    # LATTICE_LIB: a prebuilt library to load instead of building paper_2503_14688_b200/liblattice.so
    path = os.environ.get("LATTICE_LIB") or _build.build()
    if not os.path.exists(path):
        raise RuntimeError(f"CUDA library {path} is missing and could not be built")
    L = C.CDLL(path)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


STATIC_RMAX = 1024         # LATTICE_STATIC_RMAX of include/lattice.h
FLAG_BYTES = 64            # room behind a slab buffer for its 64-bit flag word (keeps 16-byte alignment)


class LatticeError(RuntimeError):
    def __init__(self, what: str, status: int, detail: str = ""):
        msg = lib().lattice_strerror(status).decode()
        super().__init__(f"{what}: {msg} ({status}){': ' + detail if detail else ''}")
        self.status = status


def _p(a: np.ndarray, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def enable_peer_access(device: int, peer_device: int) -> None:
    rc = lib().lattice_enable_peer_access(int(device), int(peer_device))
    if rc != OK:
        raise LatticeError("lattice_enable_peer_access", rc, f"{device} -> {peer_device}")


def ipc_open(handle: bytes) -> int:
    """Map another process's exportable buffer into this process; returns its device address."""
    h = (C.c_ubyte * 64).from_buffer_copy(handle)
    p = _vp()
    rc = lib().lattice_ipc_open(h, C.byref(p))
    if rc != OK:
        raise LatticeError("lattice_ipc_open", rc)
    return p.value


def ipc_close(ptr: int) -> None:
    lib().lattice_ipc_close(_vp(ptr))


def state_bytes(L: int, model: int) -> int:
    return int(lib().lattice_state_bytes(L, model))


def thresholds(model: int, delta: float, beta: float) -> np.ndarray:
    out = np.zeros(2 if model == ISING else 54, dtype=np.uint64)
    lib().lattice_thresholds(model, float(delta), float(beta), _p(out, C.c_uint64))
    return out


def thresholds64(model: int, delta: float, beta: float):
    """(thr, always) of RNG scheme 2: thresholds on the 2^64 scale."""
    n = 2 if model == ISING else 54
    thr = np.zeros(n, dtype=np.uint64)
    alw = np.zeros(n, dtype=np.uint8)
    lib().lattice_thresholds64(model, float(delta), float(beta), _p(thr, C.c_uint64), _p(alw, C.c_ubyte))
    return thr, alw


def xi(Sx, Sy, Q: int, L: int):
    Sx = np.ascontiguousarray(Sx, dtype=np.int64)
    Sy = np.ascontiguousarray(Sy, dtype=np.int64)
    rc = C.c_uint32(0)
    v = lib().lattice_xi(_p(Sx, C.c_int64), _p(Sy, C.c_int64), Sx.size, int(Q), int(L), C.byref(rc))
    return float(v), int(rc.value)


def energy(Sx, Sy, Q: int, delta: float, L: int) -> float:
    Sx = np.ascontiguousarray(Sx, dtype=np.int64)
    Sy = np.ascontiguousarray(Sy, dtype=np.int64)
    return float(lib().lattice_energy(_p(Sx, C.c_int64), _p(Sy, C.c_int64), int(Q), float(delta),
                                      int(L)))


def ubench_int_dispatch(mode: int, stream_ptr: int = 0):
    """(thread-instructions per clock per SM, elapsed ms) of the integer-dispatch micro-benchmark."""
    v, ms = C.c_double(0.0), C.c_double(0.0)
    rc = lib().lattice_ubench_int_dispatch(int(mode), _vp(stream_ptr), C.byref(v), C.byref(ms))
    if rc != OK:
        raise LatticeError("lattice_ubench_int_dispatch", rc)
    return float(v.value), float(ms.value)


def measure_buffer(L: int, model: int, rows: int, n_base: int, r_max: int, ptr: int, nbytes: int,
                   stream_ptr: int = 0):
    """(M, Q, Sx[r_max], Sy[r_max]) over base rows 0 .. n_base-1 of a caller-assembled buffer
    [colour(/plane)][rows][L/64] that is not periodic along y (include/lattice.h, lattice_view)."""
    h = _vp()
    rc = lib().lattice_view(C.byref(h), L, model, rows, _vp(ptr), nbytes, _vp(stream_ptr))
    if rc != OK:
        raise LatticeError("lattice_view", rc)
    try:
        Sx = np.zeros(r_max, dtype=np.int64)
        Sy = np.zeros(r_max, dtype=np.int64)
        M, Q = C.c_int64(0), C.c_int64(0)
        rc = lib().lattice_measure_rows(h, 0, n_base, r_max, C.byref(M), C.byref(Q),
                                        _p(Sx, C.c_int64), _p(Sy, C.c_int64))
        if rc != OK:
            raise LatticeError("lattice_measure_rows", rc)
        return int(M.value), int(Q.value), Sx, Sy
    finally:
        lib().lattice_destroy(h)


def device_copy(dst: int, src: int, nbytes: int, stream_ptr: int = 0) -> None:
    rc = lib().lattice_device_copy(_vp(dst), _vp(src), nbytes, _vp(stream_ptr))
    if rc != OK:
        raise LatticeError("lattice_device_copy", rc)


class Lattice:
    """A packed lattice in device memory (a torch.uint8 tensor owned by this object)."""

    def __init__(self, L: int, model: int = ISING, delta: float = 0.0, seed: int = 0,
                 scheme: int = 1, device: str = "cuda:0", stream=None, slab=None, exportable=False):
        """slab = (row0, n_rows) creates a row slab of the L x L lattice (include/lattice.h);
        exportable = True allocates the buffer with lattice_device_alloc so that it can be shared
        with other processes through a CUDA IPC handle (`ipc_handle`)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2503_14688_b200 needs a CUDA device; there is no CPU path")
        self.L, self.model, self.delta, self.seed = int(L), int(model), float(delta), int(seed)
        self.slab = None if slab is None else (int(slab[0]), int(slab[1]))
        if self.slab is None:
            nbytes = state_bytes(self.L, self.model)
        else:
            nbytes = int(lib().lattice_slab_bytes(self.L, self.model, self.slab[1]))
        if nbytes == 0:
            raise LatticeError("lattice_state_bytes", EINVAL, f"L={L} model={model} slab={slab}")
        self.state_nbytes = nbytes
        if self.slab is not None:
            nbytes += FLAG_BYTES                     # the slab's flag word lives behind its rows (set_flags)
        self._torch = torch
        self.device = torch.device(device)
        self._own_ptr = None
        with torch.cuda.device(self.device):
            if exportable:
                p = _vp()
                rc = lib().lattice_device_alloc(C.byref(p), nbytes)
                if rc != OK:
                    raise LatticeError("lattice_device_alloc", rc)
                self._own_ptr, self.buf = p.value, None
            else:
                self.buf = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = _vp()
            if self.slab is None:
                rc = lib().lattice_create(C.byref(h), self.L, self.model, self.delta, self.seed,
                                          _vp(self.data_ptr), nbytes, _vp(self.stream.cuda_stream))
            else:
                rc = lib().lattice_create_slab(C.byref(h), self.L, self.model, self.delta, self.seed,
                                               self.slab[0], self.slab[1], _vp(self.data_ptr),
                                               nbytes, _vp(self.stream.cuda_stream))
        if rc != OK:
            raise LatticeError("lattice_create", rc)
        self._h = h
        if scheme != 1:
            self._check(lib().lattice_set_rng_scheme(self._h, int(scheme)), "lattice_set_rng_scheme")
        self.scheme = int(scheme)

    # -- plumbing ---------------------------------------------------------------------------
    def _check(self, rc: int, what: str) -> None:
        if rc != OK:
            detail = lib().lattice_last_error(self._h).decode() if rc == ECUDA else ""
            raise LatticeError(what, rc, detail)

    @property
    def data_ptr(self) -> int:
        """Device address of the packed state."""
        return self._own_ptr if self._own_ptr is not None else self.buf.data_ptr()

    def ipc_handle(self) -> bytes:
        """64-byte CUDA IPC handle of an exportable buffer, for a neighbour in another process."""
        if self._own_ptr is None:
            raise RuntimeError("create the Lattice with exportable=True")
        h = (C.c_ubyte * 64)()
        self._check(lib().lattice_ipc_export(_vp(self._own_ptr), h), "lattice_ipc_export")
        return bytes(h)

    def close(self) -> None:
        if getattr(self, "_h", None):
            self.synchronize()
            lib().lattice_destroy(self._h)
            self._h = None
            if self._own_ptr is not None:
                lib().lattice_device_free(_vp(self._own_ptr))
                self._own_ptr = None
            self.buf = None                          # hand the device memory back to torch

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the path ---------------------------------------------------------------------------
    @property
    def time(self) -> int:
        return int(lib().lattice_time(self._h))

    @property
    def launches(self) -> int:
        return int(lib().lattice_launches(self._h))

    @property
    def specialised_launches(self) -> int:
        return int(lib().lattice_specialised_launches(self._h))

    def set_neighbours(self, up: "Lattice", down: "Lattice") -> None:
        """Row-slab mode: the slabs owning the rows above / below (self twice for a single slab)."""
        self.set_neighbour_ptrs(up.data_ptr, up.slab[1], down.data_ptr, down.slab[1])
        self._nbr = (up, down)                       # keep the neighbours' buffers alive

    def set_neighbour_ptrs(self, up_ptr: int, up_rows: int, down_ptr: int, down_rows: int) -> None:
        """The same with raw device addresses (e.g. opened from another process's IPC handle)."""
        self._check(lib().lattice_slab_set_neighbours(self._h, _vp(up_ptr), up_rows, _vp(down_ptr), down_rows),
                    "lattice_slab_set_neighbours")

    @property
    def flag_ptr(self) -> int:
        """Device address of this slab's flag word (behind its rows)."""
        return self.data_ptr + self.state_nbytes

    def set_flags(self, up_flag_ptr: int, down_flag_ptr: int) -> None:
        """Row-slab mode: order the colours on the device (include/lattice.h, lattice_slab_set_flags).
        The neighbours' flag words are `neighbour.flag_ptr` (or the address of the neighbour's buffer
        opened from its IPC handle + its slab bytes)."""
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_slab_set_flags(self._h, _vp(self.flag_ptr), _vp(up_flag_ptr), _vp(down_flag_ptr)),
                        "lattice_slab_set_flags")

    def set_time(self, t: int) -> None:
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_set_time(self._h, int(t)), "lattice_set_time")

    def sweep(self, beta) -> None:
        """Run len(beta) sweeps; beta is a host fp64 array (one entry per sweep)."""
        b = np.ascontiguousarray(np.atleast_1d(beta), dtype=np.float64)
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_sweep(self._h, b.size, _p(b, C.c_double)), "lattice_sweep")

    def sweep_record(self, beta):
        """Run len(beta) sweeps and return the r = 1 record (M, Q, S_x(1), S_y(1)) of the final state
        (lattice_sweep_record: counted inside the last white half-sweep where that kernel exists)."""
        b = np.ascontiguousarray(np.atleast_1d(beta), dtype=np.float64)
        M, Q, Sx, Sy = C.c_int64(0), C.c_int64(0), C.c_int64(0), C.c_int64(0)
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_sweep_record(self._h, b.size, _p(b, C.c_double), C.byref(M), C.byref(Q),
                                                   C.byref(Sx), C.byref(Sy)), "lattice_sweep_record")
        return int(M.value), int(Q.value), int(Sx.value), int(Sy.value)

    def half_sweep(self, colour: int, beta: float) -> None:
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_half_sweep(self._h, int(colour), float(beta)),
                        "lattice_half_sweep")

    def measure(self, r_max: int, rows=None):
        """(M, Q, Sx[r_max], Sy[r_max]) as exact integers; rows = (i0, n_rows) for a slab."""
        Sx = np.zeros(r_max, dtype=np.int64)
        Sy = np.zeros(r_max, dtype=np.int64)
        M, Q = C.c_int64(0), C.c_int64(0)
        with self._torch.cuda.device(self.device):
            if rows is None:
                rc = lib().lattice_measure(self._h, r_max, C.byref(M), C.byref(Q),
                                           _p(Sx, C.c_int64), _p(Sy, C.c_int64))
            else:
                rc = lib().lattice_measure_rows(self._h, rows[0], rows[1], r_max, C.byref(M),
                                                C.byref(Q), _p(Sx, C.c_int64), _p(Sy, C.c_int64))
        self._check(rc, "lattice_measure")
        return int(M.value), int(Q.value), Sx, Sy

    def measure_static(self, r_max: int):
        """lattice_measure_static: the same counts as measure(r_max) for r_max <= STATIC_RMAX with no
        allocation on the library side (counters in a static device array shared by all calls: do not
        overlap calls on the GPU)."""
        Sx = np.zeros(r_max, dtype=np.int64)
        Sy = np.zeros(r_max, dtype=np.int64)
        M, Q = C.c_int64(0), C.c_int64(0)
        with self._torch.cuda.device(self.device):
            rc = lib().lattice_measure_static(self._h, r_max, C.byref(M), C.byref(Q),
                                              _p(Sx, C.c_int64), _p(Sy, C.c_int64))
        if rc == EINVAL:
            raise LatticeError("lattice_measure_static", rc, lib().lattice_last_error(self._h).decode())
        self._check(rc, "lattice_measure_static")
        return int(M.value), int(Q.value), Sx, Sy

    def measure_list(self, r_list, rows=None):
        """(M, Q, Sx[len(r_list)], Sy[len(r_list)]) for a sparse list of separations r."""
        r = np.ascontiguousarray(np.asarray(r_list, dtype=np.uint32))
        Sx = np.zeros(r.size, dtype=np.int64)
        Sy = np.zeros(r.size, dtype=np.int64)
        M, Q = C.c_int64(0), C.c_int64(0)
        if rows is None:
            rows = self.slab if self.slab is not None else (0, self.L)
        with self._torch.cuda.device(self.device):
            rc = lib().lattice_measure_list(self._h, rows[0], rows[1], _p(r, C.c_uint32), r.size, C.byref(M),
                                            C.byref(Q), _p(Sx, C.c_int64), _p(Sy, C.c_int64))
        self._check(rc, "lattice_measure_list")
        return int(M.value), int(Q.value), Sx, Sy

    def get_spins(self, i0: int = 0, j0: int = 0, h: int | None = None, w: int | None = None):
        if self.slab is not None and h is None:
            i0, h = self.slab                        # a slab's default window: its own rows
        h = self.L if h is None else h
        w = self.L if w is None else w
        out = np.zeros((h, w), dtype=np.int8)
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_get_spins(self._h, i0, j0, h, w, _p(out, C.c_int8)),
                        "lattice_get_spins")
        return out

    def set_spins(self, spins, i0: int = 0, j0: int = 0) -> None:
        s = np.ascontiguousarray(spins, dtype=np.int8)
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_set_spins(self._h, i0, j0, s.shape[0], s.shape[1],
                                                _p(s, C.c_int8)), "lattice_set_spins")

    def set_measure_path(self, path: int) -> None:
        """0 automatic, 1 XOR/popcount kernels, 2 tensor cores (include/lattice.h)."""
        self._check(lib().lattice_set_measure_path(self._h, int(path)), "lattice_set_measure_path")

    def set_persist_blocks(self, max_blocks: int) -> None:
        """Cap the grid of the persistent multi-sweep kernel (0 = occupancy limit)."""
        self._check(lib().lattice_set_persist_blocks(self._h, int(max_blocks)), "lattice_set_persist_blocks")

    def fill(self, spin: int) -> None:
        """Every spin := spin (an ordered state: worst-case throughput input, tests)."""
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_fill(self._h, int(spin)), "lattice_fill")

    def synchronize(self) -> None:
        self.stream.synchronize()


class LatticeBatch:
    """n independent replicas of one lattice shape in a single device buffer (include/lattice.h,
    "Batches of independent replicas"): replica k is bit-identical to Lattice(L, model, delta,
    seeds[k]).  sweep() advances all of them; measure() returns per-replica counts."""

    def __init__(self, L: int, seeds, model: int = ISING, delta: float = 0.0, scheme: int = 1,
                 device: str = "cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2503_14688_b200 needs a CUDA device; there is no CPU path")
        self.seeds = np.ascontiguousarray(np.asarray(seeds, dtype=np.uint64))
        self.n = int(self.seeds.size)
        self.L, self.model, self.delta = int(L), int(model), float(delta)
        nbytes = int(lib().lattice_batch_bytes(self.n, self.L, self.model))
        if nbytes == 0:
            raise LatticeError("lattice_batch_bytes", EINVAL, f"n={self.n} L={L} model={model}")
        self._torch = torch
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.buf = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = _vp()
            rc = lib().lattice_create_batch(C.byref(h), self.n, self.L, self.model, self.delta,
                                            _p(self.seeds, C.c_uint64), _vp(self.buf.data_ptr()), nbytes,
                                            _vp(self.stream.cuda_stream))
        if rc != OK:
            raise LatticeError("lattice_create_batch", rc)
        self._h = h
        self.scheme = int(scheme)
        if scheme != 1:
            self._check(lib().lattice_set_rng_scheme(self._h, int(scheme)), "lattice_set_rng_scheme")

    def _check(self, rc: int, what: str) -> None:
        if rc != OK:
            detail = lib().lattice_last_error(self._h).decode() if rc == ECUDA else ""
            raise LatticeError(what, rc, detail)

    def close(self) -> None:
        if getattr(self, "_h", None):
            self.stream.synchronize()
            lib().lattice_destroy(self._h)
            self._h = None
            self.buf = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def time(self) -> int:
        return int(lib().lattice_time(self._h))

    @property
    def launches(self) -> int:
        return int(lib().lattice_launches(self._h))

    @property
    def flag_ptr(self) -> int:
        """Device address of this slab's flag word (behind its rows)."""
        return self.data_ptr + self.state_nbytes

    def set_flags(self, up_flag_ptr: int, down_flag_ptr: int) -> None:
        """Row-slab mode: order the colours on the device (include/lattice.h, lattice_slab_set_flags).
        The neighbours' flag words are `neighbour.flag_ptr` (or the address of the neighbour's buffer
        opened from its IPC handle + its slab bytes)."""
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_slab_set_flags(self._h, _vp(self.flag_ptr), _vp(up_flag_ptr), _vp(down_flag_ptr)),
                        "lattice_slab_set_flags")

    def set_time(self, t: int) -> None:
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_set_time(self._h, int(t)), "lattice_set_time")

    def sweep(self, beta) -> None:
        b = np.ascontiguousarray(np.atleast_1d(beta), dtype=np.float64)
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_sweep(self._h, b.size, _p(b, C.c_double)), "lattice_sweep")

    def half_sweep(self, colour: int, beta: float) -> None:
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_half_sweep(self._h, int(colour), float(beta)), "lattice_half_sweep")

    def fill(self, spin: int) -> None:
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_fill(self._h, int(spin)), "lattice_fill")

    def measure(self, r_max: int):
        """(M[n], Q[n], Sx[n, r_max], Sy[n, r_max]) as exact integers."""
        M = np.zeros(self.n, dtype=np.int64)
        Q = np.zeros(self.n, dtype=np.int64)
        Sx = np.zeros((self.n, r_max), dtype=np.int64)
        Sy = np.zeros((self.n, r_max), dtype=np.int64)
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_measure_batch(self._h, r_max, _p(M, C.c_int64), _p(Q, C.c_int64),
                                                    _p(Sx, C.c_int64), _p(Sy, C.c_int64)),
                        "lattice_measure_batch")
        return M, Q, Sx, Sy

    def _replica(self, k: int):
        h = _vp()
        self._check(lib().lattice_replica(self._h, int(k), C.byref(h)), "lattice_replica")
        return h

    def get_spins(self, k: int, i0: int = 0, j0: int = 0, h: int | None = None, w: int | None = None):
        h = self.L if h is None else h
        w = self.L if w is None else w
        out = np.zeros((h, w), dtype=np.int8)
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_get_spins(self._replica(k), i0, j0, h, w, _p(out, C.c_int8)),
                        "lattice_get_spins")
        return out

    def set_spins(self, k: int, spins, i0: int = 0, j0: int = 0) -> None:
        s = np.ascontiguousarray(spins, dtype=np.int8)
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_set_spins(self._replica(k), i0, j0, s.shape[0], s.shape[1],
                                                _p(s, C.c_int8)), "lattice_set_spins")

    def measure_replica(self, k: int, r_max: int, rows=None):
        Sx = np.zeros(r_max, dtype=np.int64)
        Sy = np.zeros(r_max, dtype=np.int64)
        M, Q = C.c_int64(0), C.c_int64(0)
        i0, n = (0, self.L) if rows is None else rows
        with self._torch.cuda.device(self.device):
            self._check(lib().lattice_measure_rows(self._replica(k), i0, n, r_max, C.byref(M), C.byref(Q),
                                                   _p(Sx, C.c_int64), _p(Sy, C.c_int64)), "lattice_measure_rows")
        return int(M.value), int(Q.value), Sx, Sy

    def synchronize(self) -> None:
        self.stream.synchronize()
