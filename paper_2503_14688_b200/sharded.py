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


# ---- one process per GPU ---------------------------------------------------------------------
def neighbour_ranks(rank: int, world: int):
    """(up, down): the ranks that own the rows above / below rank's slab (periodic)."""
    return (rank - 1) % world, (rank + 1) % world


def exchange_handles(my_handle: bytes, group=None):
    """All-gather the 64-byte IPC handles over torch.distributed (any backend) and return
    (handle of the upper neighbour, handle of the lower neighbour)."""
    import torch.distributed as dist
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    handles = [None] * world
    dist.all_gather_object(handles, bytes(my_handle), group=group)
    if any(h is None or len(h) != 64 for h in handles):
        raise RuntimeError("a rank did not contribute a 64-byte handle")
    up, down = neighbour_ranks(rank, world)
    return handles[up], handles[down]


class SlabRank:
    """This process's slab of an L x L lattice sharded over the ranks of a torch.distributed
    group, one rank per GPU.  Buffers are shared through CUDA IPC handles, so the half-sweep
    kernel of each rank writes its boundary rows straight into its neighbours' halo rows
    (NVLink P2P); the only collectives are the barrier that orders the colours and the u64
    all-reduce of the measurement counts."""

    def __init__(self, L: int, seed: int = 0, model: int = lat.ISING, delta: float = 0.0,
                 device: str = "cuda:0", group=None):
        import torch
        import torch.distributed as dist
        self._torch, self._dist, self.group = torch, dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        if L % self.world:
            raise ValueError("the number of ranks must divide L")
        rows = L // self.world
        self.L, self.rows = L, rows
        self.lat = lat.Lattice(L, model, delta, seed, device=device, slab=(self.rank * rows, rows),
                               exportable=True)
        self._opened = []
        if self.world == 1:
            self.lat.set_neighbours(self.lat, self.lat)
        else:
            h_up, h_down = exchange_handles(self.lat.ipc_handle(), group)
            with torch.cuda.device(self.lat.device):
                p_up = lat.ipc_open(h_up)
                p_down = p_up if self.world == 2 else lat.ipc_open(h_down)   # one mapping per buffer
            self._opened = [p_up] if self.world == 2 else [p_up, p_down]
            self.lat.set_neighbour_ptrs(p_up, rows, p_down, rows)
        self._t = 0
        self._fence()

    def _fence(self) -> None:
        self.lat.synchronize()
        if self.world > 1:
            self._dist.barrier(self.group)

    @property
    def time(self) -> int:
        return self._t

    def sweep(self, beta) -> None:
        for b in np.atleast_1d(np.asarray(beta, dtype=np.float64)):
            for colour in (0, 1):
                self.lat.half_sweep(colour, float(b))
                self._fence()                        # every rank's mirrors have landed
            self._t += 1
            self.lat.set_time(self._t)

    def measure(self):
        """(M, Q, S_x(1), S_y(1)) of the whole lattice on every rank."""
        M, Q, Sx, Sy = self.lat.measure(1)
        t = self._torch.tensor([M, Q, int(Sx[0]), int(Sy[0])], dtype=self._torch.int64)
        if self.world > 1:
            if self._dist.get_backend(self.group) == "nccl":
                t = t.to(self.lat.device)
            self._dist.all_reduce(t, op=self._dist.ReduceOp.SUM, group=self.group)
        return tuple(int(x) for x in t.cpu())

    def get_spins(self) -> np.ndarray:
        """This rank's own rows."""
        return self.lat.get_spins()

    def close(self) -> None:
        self._fence()
        for p in self._opened:
            lat.ipc_close(p)
        self._opened = []
        self.lat.close()
