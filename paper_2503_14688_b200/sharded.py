"""Row-slab domain decomposition: one L x L lattice spread over several slabs / GPUs.

The paper's third level of parallelism.  Each slab
owns L / n consecutive rows plus one halo row above and below (include/lattice.h, "Row-slab
domain decomposition").  There is no separate exchange step: the half-sweep kernel of a slab
stores its first and last own row a second time straight into the neighbours' halo rows -- plain
stores (and atomics for late tie flips) to pointers that are peer-GPU memory when the slabs sit on
different devices (NVLink P2P through NVSwitch), so the transfer rides on the update kernel.
What this driver adds is ordering: every slab finishes colour c before any slab starts colour
1 - c (stream order on one device, events across devices).

`ShardedLattice`: one process drives all devices of the node (peer access enabled explicitly);
`SlabRank`: one process per GPU.  Random numbers are keyed by global (row, column): the result is bit-identical to the
unsharded lattice for any number of slabs (tests/test_gpu_sharded.py).
"""
from __future__ import annotations

import numpy as np

from . import binding as lat


class ShardedLattice:
    def __init__(self, L: int, n_slabs: int, seed: int = 0, devices=None, model: int = lat.ISING,
                 delta: float = 0.0, device_flags: bool = False):
        """device_flags = True: the colours are ordered on the device (lattice_slab_set_flags: every
        half-sweep launch waits for the neighbours' published counts) instead of by stream order /
        events from the host."""
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
            for nb in (up, down):                     # kernels of s store into nb's halo rows
                if nb.device != s.device:
                    lat.enable_peer_access(s.device.index, nb.device.index)
            s.set_neighbours(up, down)
        self.device_flags = bool(device_flags)
        if self.device_flags:
            for k, s in enumerate(self.slabs):
                s.set_flags(self.slabs[(k - 1) % n_slabs].flag_ptr, self.slabs[(k + 1) % n_slabs].flag_ptr)
        self._t = 0
        self.synchronize()                            # every slab has published its count before any sweep

    # -- ordering -------------------------------------------------------------------------------
    def _fence(self) -> None:
        """All slabs have finished (and mirrored) the colour just launched before the next starts."""
        if self.device_flags:
            return                                    # ordered on the device (slab_flags.cuh)
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

    def measure(self, r_max: int = 1):
        """Whole-lattice counts, the slabs' partial sums added up: (M, Q, S_x(1), S_y(1)) for
        r_max == 1 (one pass per slab), else (M, Q, Sx[r_max], Sy[r_max]): every slab measures a
        temporary buffer of its own rows followed by the next r_max rows of the lattice."""
        if r_max == 1:
            tot = np.zeros(4, dtype=np.int64)
            for s in self.slabs:
                M, Q, Sx, Sy = s.measure(1)
                tot += np.array([M, Q, Sx[0], Sy[0]], dtype=np.int64)
            return tuple(int(x) for x in tot)
        torch = self._torch
        rows = self.L // self.n
        wpr = self.L // 64
        planes = 2 if self.model == lat.ISING else 4
        M = Q = 0
        Sx = np.zeros(r_max, dtype=np.int64)
        Sy = np.zeros(r_max, dtype=np.int64)
        self.synchronize()
        for k, s in enumerate(self.slabs):
            # own rows, then r_max rows from the slabs below (possibly several, periodic)
            pieces = []
            for p in range(planes):
                own = s.buf[:s.state_nbytes].view(planes, rows + 2, wpr * 4)[p, 1:rows + 1]
                ext, need, j = [own], r_max, k
                while need > 0:
                    j = (j + 1) % self.n
                    nb = self.slabs[j].buf[:self.slabs[j].state_nbytes].view(planes, rows + 2, wpr * 4)[p, 1:1 + min(need, rows)]
                    ext.append(nb.to(s.device))
                    need -= min(need, rows)
                pieces.append(torch.cat(ext, dim=0))
            with torch.cuda.device(s.device):
                buf = torch.stack(pieces, dim=0).contiguous()
                torch.cuda.current_stream(s.device).synchronize()
                m, q, sx, sy = lat.measure_buffer(self.L, self.model, rows + r_max, rows, r_max,
                                                  buf.data_ptr(), buf.numel(), s.stream.cuda_stream)
            M += m; Q += q; Sx += sx; Sy += sy
        return M, Q, Sx, Sy

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
                 device: str = "cuda:0", group=None, device_flags: bool = False):
        """device_flags = True: no barrier per half-sweep; the ranks' kernels wait for each other's
        published counts (lattice_slab_set_flags).  For one rank per PHYSICAL GPU only: ranks that
        share a GPU must not run kernels that wait on one another."""
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
            self._down_ptr = p_down
            self.lat.set_neighbour_ptrs(p_up, rows, p_down, rows)
        self.device_flags = bool(device_flags)
        if self.device_flags:
            nb = self.lat.state_nbytes                # every rank's slab has the same size
            if self.world == 1:
                self.lat.set_flags(self.lat.flag_ptr, self.lat.flag_ptr)
            else:
                self.lat.set_flags(p_up + nb, p_down + nb)
        self._t = 0
        self._fence()                                 # every rank has published its count

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
                if not self.device_flags:
                    self._fence()                    # every rank's mirrors have landed
            self._t += 1
            self.lat.set_time(self._t)

    def _all_reduce(self, values):
        t = self._torch.tensor(values, dtype=self._torch.int64)
        if self.world > 1:
            if self._dist.get_backend(self.group) == "nccl":
                t = t.to(self.lat.device)
            self._dist.all_reduce(t, op=self._dist.ReduceOp.SUM, group=self.group)
        return t.cpu().numpy()

    def measure(self, r_max: int = 1):
        """Whole-lattice counts on every rank: (M, Q, S_x(1), S_y(1)) for r_max == 1, else
        (M, Q, Sx[r_max], Sy[r_max]) with r_max <= rows per rank (the partner rows come from the
        lower neighbour's buffer through its IPC mapping)."""
        if r_max == 1:
            M, Q, Sx, Sy = self.lat.measure(1)
            return tuple(int(x) for x in self._all_reduce([M, Q, int(Sx[0]), int(Sy[0])]))
        if r_max > self.rows:
            raise ValueError("r_max must not exceed the rows per rank")
        rows, wpr = self.rows, self.L // 64
        planes = 2 if self.lat.model == lat.ISING else 4
        row_bytes, plane_bytes = wpr * 4, (rows + 2) * wpr * 4
        ext_rows = rows + r_max
        nbytes = planes * ext_rows * row_bytes
        down = self._down_ptr if self.world > 1 else self.lat.data_ptr
        self._fence()                                 # every rank's state is final
        with self._torch.cuda.device(self.lat.device):
            buf = self._torch.empty(nbytes, dtype=self._torch.uint8, device=self.lat.device)
            st = self.lat.stream.cuda_stream
            for p in range(planes):
                dst = buf.data_ptr() + p * ext_rows * row_bytes
                lat.device_copy(dst, self.lat.data_ptr + p * plane_bytes + row_bytes, rows * row_bytes, st)
                lat.device_copy(dst + rows * row_bytes, down + p * plane_bytes + row_bytes,
                                r_max * row_bytes, st)
            M, Q, Sx, Sy = lat.measure_buffer(self.L, self.lat.model, ext_rows, rows, r_max,
                                              buf.data_ptr(), nbytes, st)
        self._fence()                                 # neighbours may sweep again
        tot = self._all_reduce([M, Q] + Sx.tolist() + Sy.tolist())
        return int(tot[0]), int(tot[1]), tot[2:2 + r_max].copy(), tot[2 + r_max:].copy()

    def get_spins(self) -> np.ndarray:
        """This rank's own rows."""
        return self.lat.get_spins()

    def close(self) -> None:
        self._fence()
        for p in self._opened:
            lat.ipc_close(p)
        self._opened = []
        self.lat.close()
