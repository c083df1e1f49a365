"""Row-slab domain decomposition: one L x L lattice spread over several slabs / GPUs.

The paper's third level of parallelism.  Each slab
owns L / n consecutive rows plus one halo row above and below (include/lattice.h, "Row-slab
domain decomposition").  There is no separate exchange step: the half-sweep kernel of a slab
stores its first and last own row a second time straight into the neighbours' halo rows -- plain
stores (and atomics for late tie flips) to pointers that are peer-GPU memory when the slabs sit on
different devices (NVLink P2P through NVSwitch), so the transfer rides on the update kernel.
What this driver adds is ordering: every slab finishes colour c before any slab starts colour
1 - c (stream order on one device, events across devices).

One process drives all devices of the node (torch enables peer access on the first cross-device
copy).  Random numbers are keyed by global (row, column): the result is bit-identical to the
unsharded lattice for any number of slabs (tests/test_gpu_sharded.py).
"""
from __future__ import annotations

import numpy as np

from . import binding as lat


class ShardedLattice:
    def __init__(self, L: int, n_slabs: int, seed: int = 0, devices=None, model: int = lat.ISING,
                 delta: float = 0.0):
        import torch
        if n_slabs < 1 or L % n_slabs:
            raise ValueError("n_slabs must divide L")
        rows = L // n_slabs
        devices = list(devices) if devices else ["cuda:0"] * n_slabs
        if len(devices) != n_slabs:
            raise ValueError("one device per slab")
        self.L, self.model, self.delta, self.seed, self.n = L, model, delta, seed, n_slabs
        self._torch = torch
        self.slabs = [lat.Lattice(L, model, delta, seed, device=d, slab=(k * rows, rows))
                      for k, d in enumerate(devices)]
        self._multi_device = len({str(s.device) for s in self.slabs}) > 1
        for k, s in enumerate(self.slabs):
            up, down = self.slabs[(k - 1) % n_slabs], self.slabs[(k + 1) % n_slabs]
            if self._multi_device:
                for nb in (up, down):                 # one tiny copy makes torch enable peer access
                    if nb.device != s.device:
                        s.buf[:16].copy_(nb.buf[:16].to(s.device, copy=True) * 0 + s.buf[:16])
            s.set_neighbours(up, down)
        self._t = 0
        self.synchronize()

    # -- ordering -------------------------------------------------------------------------------
    def _fence(self) -> None:
        """All slabs have finished (and mirrored) the colour just launched before the next starts."""
        if not self._multi_device:
            streams = {s.stream.cuda_stream for s in self.slabs}
            if len(streams) == 1:
                return                                # one stream: launch order is enough
        torch = self._torch
        events = []
        for s in self.slabs:
            with torch.cuda.device(s.device):
                e = torch.cuda.Event()
                e.record(s.stream)
                events.append(e)
        for k, s in enumerate(self.slabs):
            for nb in ((k - 1) % self.n, (k + 1) % self.n):
                if nb != k:
                    s.stream.wait_event(events[nb])

    def synchronize(self) -> None:
        for s in self.slabs:
            s.synchronize()

    # -- the path -------------------------------------------------------------------------------
    @property
    def time(self) -> int:
        return self._t

    def sweep(self, beta) -> None:
        for b in np.atleast_1d(np.asarray(beta, dtype=np.float64)):
            for colour in (0, 1):
                for s in self.slabs:
                    s.half_sweep(colour, float(b))
                self._fence()
            self._t += 1
            for s in self.slabs:
                s.set_time(self._t)

    def measure(self):
        """(M, Q, S_x(1), S_y(1)) of the whole lattice: the slabs' partial sums added up."""
        tot = np.zeros(4, dtype=np.int64)
        for s in self.slabs:
            M, Q, Sx, Sy = s.measure(1)
            tot += np.array([M, Q, Sx[0], Sy[0]], dtype=np.int64)
        return tuple(int(x) for x in tot)

    def get_spins(self) -> np.ndarray:
        return np.concatenate([s.get_spins() for s in self.slabs], axis=0)

    def close(self) -> None:
        for s in self.slabs:
            s.close()
