"""The N > 1 mode is "replicas only": no data-path collective, only the
plumbing around the timed region.  World-size-2 gloo processes on CPU exercise that plumbing."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
from paper_2503_14688_b200 import replicas
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
# before init: single-process behaviour
assert replicas.agree_min(4096) == 4096 and replicas.max_over_ranks(1.5) == 1.5
dist.init_process_group("gloo", rank=rank, world_size=world)
seeds = [replicas.replica_seed(2503146884, r) for r in range(world)]
assert len(set(seeds)) == world and seeds[0] == 2503146884
# ranks propose different sizes (rank 1 has less free memory): all agree on the smaller
L = replicas.agree_min(1 << (20 - rank))
assert L == 1 << (20 - (world - 1)), L
replicas.barrier()
# rank r took (100 + 10 r) ms: the job took the slowest rank's time
ms = replicas.max_over_ranks(100.0 + 10.0 * rank)
assert ms == 100.0 + 10.0 * (world - 1), ms
rate = replicas.job_rate(L * L * 16, world, ms)
assert abs(rate - world * L * L * 16 / (ms * 1e6)) < 1e-9
replicas.barrier()
dist.destroy_process_group()
print("ok", rank)
'''


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_replica_plumbing_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for rank, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, out
        assert f"ok {rank}" in out


def test_single_process_defaults():
    from paper_2503_14688_b200 import replicas
    assert replicas.agree_min(123) == 123
    assert replicas.max_over_ranks(2.5) == 2.5
    replicas.barrier()
    assert replicas.job_rate(10 ** 12, 1, 250.0) == 4000.0
    assert replicas.replica_seed(7, 3) == 3007


SHARD_WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
from paper_2503_14688_b200 import sharded
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
assert sharded.neighbour_ranks(0, 4) == (3, 1) and sharded.neighbour_ranks(3, 4) == (2, 0)
assert sharded.neighbour_ranks(0, 1) == (0, 0)
# every rank contributes a (fake) 64-byte IPC handle; each gets its two neighbours' handles back
mine = bytes([rank]) * 64
up, down = sharded.exchange_handles(mine)
u, d = sharded.neighbour_ranks(rank, world)
assert up == bytes([u]) * 64 and down == bytes([d]) * 64
try:
    sharded.exchange_handles(b"short")
    raise SystemExit("a short handle must be rejected")
except RuntimeError:
    pass
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
'''


def test_sharded_handle_exchange_world_size_2_gloo(tmp_path):
    """Row-slab mode, one process per GPU: the IPC-handle exchange that wires the neighbours'
    halo pointers (the CUDA part runs in tests/test_gpu_sharded.py)."""
    script = tmp_path / "shard_worker.py"
    script.write_text(SHARD_WORKER)
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for rank, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, out
        assert f"ok {rank}" in out
