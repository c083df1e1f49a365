"""Row-slab domain decomposition (include/lattice.h): N slabs with fused halo mirroring evolve
bit for bit like the whole lattice and like the oracle.  All slabs sit on one GPU here (the
mirror pointers are then ordinary device memory; across GPUs they are NVLink peer pointers)."""
import numpy as np
import pytest

import oracle
import paper_2503_14688_b200 as lat
from paper_2503_14688_b200 import workloads
from paper_2503_14688_b200.sharded import ShardedLattice

pytestmark = pytest.mark.gpu
BETA_C = workloads.BETA_C_ISING


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
@pytest.mark.parametrize("L,n_slabs", [(256, 1), (256, 2), (256, 4), (1024, 2), (1024, 16), (2048, 8)])
def test_sharded_equals_unsharded_and_oracle(L, n_slabs, model):
    seed = 777 + L + n_slabs
    sh = ShardedLattice(L, n_slabs, seed, model=model)
    g = lat.Lattice(L, model, 0.0, seed)
    assert np.array_equal(sh.get_spins(), g.get_spins())            # the disordered start
    bc = BETA_C if model == lat.ISING else workloads.BETA_BC
    beta = [bc] * 6 + [0.0, 0.3, 5.0, np.inf] + [bc / 1.01] * 6
    sh.sweep(beta)
    g.sweep(beta)
    assert sh.time == g.time == len(beta)
    assert np.array_equal(sh.get_spins(), g.get_spins())
    M, Q, Sx, Sy = g.measure(1)
    assert sh.measure() == (M, Q, int(Sx[0]), int(Sy[0]))
    # C(r) for r > 1: own rows + the next r_max rows of the lattice, per slab (r_max may span slabs)
    for r_max in (2, 37, min(L // 2, L // n_slabs + 5)):
        Mg, Qg, Sxg, Syg = g.measure(r_max)
        Ms, Qs, Sxs, Sys = sh.measure(r_max)
        assert (Ms, Qs) == (Mg, Qg) and np.array_equal(Sxs, Sxg) and np.array_equal(Sys, Syg), r_max
    if L <= 1024:
        o = oracle.OracleLattice(L, model, 0.0, seed)
        o.sweep(beta)
        assert np.array_equal(sh.get_spins(), o.get_spins())
    # halos are the neighbours' boundary rows (the mirror stores and the late tie flips landed)
    rows = L // n_slabs
    for k, s in enumerate(sh.slabs):
        own = s.get_spins()
        up_last = sh.slabs[(k - 1) % n_slabs].get_spins()[-1]
        dn_first = sh.slabs[(k + 1) % n_slabs].get_spins()[0]
        assert np.array_equal(s.get_spins((k * rows - 1) % L, 0, 1, L)[0], up_last)
        assert np.array_equal(s.get_spins((k * rows + rows) % L, 0, 1, L)[0], dn_first)
        assert own.shape == (rows, L)
    sh.close(); g.close()


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
def test_sharded_many_sweeps_many_ties_across_boundaries(model):
    """Long enough that hundreds of tied lanes fall on mirrored boundary rows."""
    L, n_slabs, seed = 512, 8, 31337
    sh = ShardedLattice(L, n_slabs, seed, model=model)
    g = lat.Lattice(L, model, 0.0, seed)
    bc = BETA_C if model == lat.ISING else workloads.BETA_BC
    for _ in range(5):
        sh.sweep([bc] * 40)
        g.sweep([bc] * 40)
        assert np.array_equal(sh.get_spins(), g.get_spins())
    sh.close(); g.close()


@pytest.mark.parametrize("delta,T", [(0.7, 1.2), (-1.3, 2.0), (1.965, 0.6)])
def test_sharded_blume_capel_with_crystal_field(delta, T):
    """Slab mode for Delta != 0 (the general marching kernel mirrors halos and late tie flips too)."""
    L, n_slabs, seed = 512, 4, 2718
    sh = ShardedLattice(L, n_slabs, seed, model=lat.BLUME_CAPEL, delta=delta)
    o = oracle.OracleLattice(L, lat.BLUME_CAPEL, delta, seed)
    beta = [1.0 / T] * 30 + [0.0, 3.0] + [1.0 / T] * 8
    sh.sweep(beta)
    o.sweep(beta)
    assert np.array_equal(sh.get_spins(), o.get_spins())
    M, Q, Sx, Sy = o.measure(1)
    assert sh.measure() == (M, Q, int(Sx[0]), int(Sy[0]))
    sh.close(); o.close()


def _n_gpus():
    import torch
    return torch.cuda.device_count()


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
def test_sharded_across_physical_devices(model):
    """The multi-device mode on real peers (skipped on a 1-GPU box, which is all this project has been
    run on): one slab per GPU, halo rows and late tie flips stored straight into the neighbour GPU's
    memory (peer pointers, atomicXor_system), bit-identical to the unsharded lattice."""
    n = _n_gpus()
    if n < 2:
        pytest.skip("needs >= 2 CUDA devices with peer access")
    n = min(n, 4)
    L, seed = 1024, 4711
    sh = ShardedLattice(L, n, seed, devices=[f"cuda:{k}" for k in range(n)], model=model)
    g = lat.Lattice(L, model, 0.0, seed)
    bc = BETA_C if model == lat.ISING else workloads.BETA_BC
    for _ in range(3):
        sh.sweep([bc] * 30)
        g.sweep([bc] * 30)
        assert np.array_equal(sh.get_spins(), g.get_spins())
    M, Q, Sx, Sy = g.measure(1)
    assert sh.measure() == (M, Q, int(Sx[0]), int(Sy[0]))
    sh.close(); g.close()


@pytest.mark.parametrize("model", [lat.ISING, lat.BLUME_CAPEL])
def test_device_side_flags_order_the_colours(model):
    """lattice_slab_set_flags: every half-sweep launch is wait kernel + marching kernel + publish kernel.
    All slabs share one device and one stream here, so the neighbours' counts are always there when a
    wait kernel runs (a wait that really spins must not be run on one GPU: B200_PROFILING.md); what is
    checked is the published arithmetic, the launch sequence and that nothing else changes: spins equal
    the host-ordered sharded lattice, the unsharded one and the oracle."""
    import torch
    L, n = 1024, 4
    beta = BETA_C if model == lat.ISING else workloads.BETA_BC
    sh = ShardedLattice(L, n, seed=99, model=model, device_flags=True)
    ho = ShardedLattice(L, n, seed=99, model=model)
    o = oracle.OracleLattice(L, model, 0.0, 99)
    sched = [beta] * 5 + [0.0, beta, 0.7 * beta]
    n0 = sh.slabs[0].launches
    sh.sweep(sched)
    ho.sweep(sched)
    o.sweep(sched)
    # per sweep and slab: 2 x (wait + march + publish) + the publish of set_time
    assert sh.slabs[0].launches - n0 == len(sched) * 7
    sh.synchronize()
    for s in sh.slabs:
        flag = s.buf[s.state_nbytes:s.state_nbytes + 8].view(torch.int64).item()
        assert flag == 2 * len(sched)
    want = o.get_spins()
    assert np.array_equal(sh.get_spins(), want)
    assert np.array_equal(ho.get_spins(), want)
    assert sh.measure(1) == ho.measure(1)
    # a checkpoint-style time change republishes the count
    for d in (sh, ho):
        for s in d.slabs:
            s.set_time(100)
        d._t = 100
        d.sweep([beta] * 2)
    sh.synchronize()
    assert sh.slabs[2].buf[sh.slabs[2].state_nbytes:sh.slabs[2].state_nbytes + 8].view(torch.int64).item() == 204
    assert np.array_equal(sh.get_spins(), ho.get_spins())
    sh.close(); ho.close(); o.close()


def test_slab_api_errors():
    L = 256
    with pytest.raises(lat.LatticeError):
        lat.Lattice(L, lat.ISING, 0.0, 1, slab=(0, 100))             # n_rows not a multiple of 64
    with pytest.raises(lat.LatticeError):
        lat.Lattice(L, lat.ISING, 0.0, 1, slab=(32, 64))             # row0 not a multiple of 64
    b = lat.Lattice(L, lat.BLUME_CAPEL, 4.7, 1, slab=(0, 256))      # |Delta| > 4: no marching table
    b.set_neighbours(b, b)
    with pytest.raises(lat.LatticeError):
        b.half_sweep(0, 0.5)
    b.close()
    s = lat.Lattice(L, lat.ISING, 0.0, 1, slab=(64, 128))
    with pytest.raises(lat.LatticeError) as e:
        s.half_sweep(0, 0.4)                                         # neighbours not set
    assert e.value.status == lat.binding.ESTATE
    with pytest.raises(lat.LatticeError):
        s.measure(2)                                                 # only r_max = 1 on a slab
    with pytest.raises(lat.LatticeError):
        s.get_spins(0, 0, 8, L)                                      # rows outside the slab
    assert s.get_spins().shape == (128, L)
    assert s.get_spins(63, 0, 130, L).shape == (130, L)              # own rows and both halos
    s.close()


RANK_WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np
import torch.distributed as dist
import paper_2503_14688_b200 as lat
from paper_2503_14688_b200 import sharded, workloads
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
L, model, seed = int(sys.argv[2]), int(sys.argv[3]), 4711
dist.init_process_group("gloo", rank=rank, world_size=world)
beta = [workloads.BETA_C_ISING if model == 0 else workloads.BETA_BC] * 12 + [0.0, 0.7]
s = sharded.SlabRank(L, seed, model)
s.sweep(beta)
counts = s.measure()
corr = s.measure(40)
parts = [None] * world
dist.all_gather_object(parts, s.get_spins())
if rank == 0:
    g = lat.Lattice(L, model, 0.0, seed)
    g.sweep(beta)
    assert np.array_equal(np.concatenate(parts, axis=0), g.get_spins())
    M, Q, Sx, Sy = g.measure(1)
    assert counts == (M, Q, int(Sx[0]), int(Sy[0])), (counts, M, Q, Sx, Sy)
    M, Q, Sx, Sy = g.measure(40)
    assert corr[0] == M and corr[1] == Q and np.array_equal(corr[2], Sx) and np.array_equal(corr[3], Sy)
    g.close()
s.close()
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
'''


@pytest.mark.parametrize("world,L,model", [(2, 512, lat.ISING), (3, 768, lat.ISING), (2, 512, lat.BLUME_CAPEL)])
def test_one_process_per_slab_through_cuda_ipc(tmp_path, world, L, model):
    """One process per slab (as one process per GPU would run it), neighbours' halo rows reached
    through CUDA IPC handles exchanged over torch.distributed (gloo), colours ordered by
    barriers.  All processes share this box's single GPU; no kernel waits on another process."""
    import os, socket, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "rank_worker.py"
    script.write_text(RANK_WORKER)
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script), root, str(L), str(model)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=300)[0] for p in procs]
    for rank, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, out
        assert f"ok {rank}" in out
