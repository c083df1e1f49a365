#!/usr/bin/env python
"""bench.py -- spin updates/ns of the checkerboard Metropolis sweep on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

A "step" is one full-lattice Metropolis sweep (black half-sweep + white half-sweep, thresholds
rebuilt from the step's beta on the host) of BASELINE.json's throughput configuration:
2D Ising, L = 2^20 (128 GiB at 1 bit/spin), disordered start, beta_c.  If the device cannot
hold 128 GiB the largest power-of-two L that fits is used and named in config.workload.

One JSON line is printed by rank 0:
  value     whole-job spin updates/ns, device-timed (CUDA events), lattice resident in HBM
  e2e       the same metric through the C-ABI with host buffers every step: the step's beta goes
            in as a host fp64 array and the step's result (M, Q, S_x(1), S_y(1) -> e, m) comes
            back to host memory (lattice_sweep + lattice_measure), all inside the timed region
  roofline  the binding roofline of the dominant kernel (the half-sweep): "bound": "alu" -- thread-
            instructions of the 16-lane integer dispatch class per launch / mean launch time,
            against 148 SM x 64 lanes x the sampled SM clock
  roofline_hbm  the HBM roofline BASELINE.json's metric asks for: algorithmic bytes (0.375
            B/update Ising, 0.75 BC: read both colours once, write one) / mean launch time,
            against the measured copy bandwidth in MEASURED_PEAKS.json
  cpu_baseline  the oracle, as it stands, on the host cores over a bounded sample
  measure   the measurement pass (M, Q, C(r) on both axes) timed separately after the sweeps

N > 1 (torchrun): the path is specified for one GPU with no collectives (BASELINE.json
north_star), so every rank runs an independent replica (own seed) -- "replicas only", weak
scaling; time is the max over ranks, value the sum of updates over ranks / that time.

--impl reference times the CPU oracle on the same metric (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2503_14688_b200 import workloads  # noqa: E402

METRIC = "spin updates/ns per B200 (Ising & Blume-Capel) and % of HBM roofline"
UNIT = "spin updates/ns"
BYTES_PER_UPDATE = {workloads.ISING: 0.375, workloads.BLUME_CAPEL: 0.75}
# Integer-pipe roofline of the dominant kernel: thread-instructions of the
# half-rate class (ALU pipe: LOP3/SHF/SEL/ISETP..., plus IMAD.WIDE/IMAD.HI, which block the same
# 16-lane dispatch for two cycles) per spin update.
#   ALGORITHMIC: the floor of the method under the RNG contract (folded Philox planes, 2 LOP3 per
#   word per plane of compare, class logic, 2^-8 tails), the analogue of algorithmic bytes;
#   EXECUTED: from the committed ncu captures under profiles/ (sm__inst_executed_pipe_alu +
#   IMAD.WIDE/HI counts / updates per launch).
ALG_HALF_RATE_INSTR_PER_UPDATE = {workloads.ISING: 2.98, workloads.BLUME_CAPEL: 4.46}
EXE_HALF_RATE_INSTR_PER_UPDATE = {workloads.ISING: 3.39, workloads.BLUME_CAPEL: 5.30}
#: DRAM bytes per update measured by ncu (dram__bytes_read.sum + dram__bytes_write.sum) / updates
DRAM_BYTES_PER_UPDATE_NCU = {workloads.ISING: 0.383, workloads.BLUME_CAPEL: 0.667}
SM_COUNT, HALF_RATE_LANES_PER_CLK_PER_SM = 148, 64
KERNEL = {workloads.ISING: "ising_march_kernel", workloads.BLUME_CAPEL: "bc_march_kernel"}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(p.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


class ClockSampler:
    """nvidia-smi clock/throttle samples during the timed region (profiling recipe's line)."""
    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1])); mx.append(float(f[2]))
                except ValueError:
                    continue
                for name, v in zip(names, f[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def oracle_rate(w, L, sweeps, scheme=1):
    """Updates/ns of the CPU oracle (all host cores) on `sweeps` sweeps of an L x L sample."""
    import oracle
    oracle.build()
    cores = os.cpu_count() or 1
    oracle.set_threads(cores)
    o = oracle.OracleLattice(L, w.model, w.delta, w.seed, scheme)
    beta = w.beta_schedule(sweeps)
    t0 = time.perf_counter()
    o.sweep(beta)
    dt = time.perf_counter() - t0
    o.close()
    return L * L * sweeps / dt / 1e9, dt, oracle.get_threads()


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, same metric and config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workloads.CONFIGS[args.workload]
    Ls, ns = min(w.L, 4096), 8                   # one step = 8 sweeps of a 4096 x 4096 sample (~1 s)
    for _ in range(args.warmup):
        oracle_rate(w, 256, 1)
    t0 = time.perf_counter()
    rates = [oracle_rate(w, Ls, ns) for _ in range(args.steps)]
    wall = time.perf_counter() - t0
    value = Ls * Ls * ns * args.steps / sum(r[1] for r in rates) / 1e9
    sample = (f"{args.steps} steps, each {ns} sweeps of a {Ls}x{Ls} {w.name}-shaped lattice "
              f"(same model, beta, RNG scheme 1)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32",
        "data": "synthetic", "config": {"workload": w.name, "L": w.L, "sample_L": Ls},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": rates[0][2] if rates else 0,
                         "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def run_sharded(args):
    """One L x L lattice in row slabs, one rank per GPU: the optional
    strong-scaling mode.  The default N > 1 mode stays independent replicas."""
    import torch
    import torch.distributed as dist
    from paper_2503_14688_b200 import replicas
    from paper_2503_14688_b200.sharded import SlabRank

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0")) % max(torch.cuda.device_count(), 1)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29533")
    if args.dist_backend == "nccl":
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    else:
        dist.init_process_group("gloo", rank=rank, world_size=world)
    w = workloads.CONFIGS[args.workload]
    L = args.L or w.L
    free, _ = torch.cuda.mem_get_info(dev)
    per_spin = 8 if w.model == workloads.ISING else 4
    while L > 256 * world and L * L // per_spin // world > free - (2 << 30):
        L //= 2
    L = replicas.agree_min(L, dev if args.dist_backend == "nccl" else "cpu")
    s = SlabRank(L, w.seed, w.model, w.delta, device=str(dev))
    sched = w.beta_schedule(args.warmup + args.steps)
    s.sweep(sched[:args.warmup])
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    dist.barrier()
    n0 = s.lat.launches
    ev0.record(s.lat.stream)
    s.sweep(sched[args.warmup:])
    ev1.record(s.lat.stream)
    launches = s.lat.launches - n0
    torch.cuda.synchronize(dev)
    ms = replicas.max_over_ranks(ev0.elapsed_time(ev1), dev if args.dist_backend == "nccl" else "cpu")
    counts = s.measure()
    if rank == 0:
        line = {"metric": METRIC, "value": L * L * args.steps / (ms * 1e6), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "u32",
                "data": "synthetic",
                "config": {"workload": w.name if L == w.L else f"{w.name}@L={L}", "L": L,
                           "parallelism": f"row slabs x{world}, halo rows mirrored by the update kernel",
                           "rows_per_rank": L // world},
                "gpu_launches": int(launches),
                "record": {"M": counts[0], "Q": counts[1], "Sx1": counts[2], "Sy1": counts[3]}}
        print(json.dumps(line))
    s.close()
    dist.destroy_process_group()


def pick_L(w, torch, dev):
    """Largest power-of-two L <= w.L whose packed state fits in the free device memory."""
    free, _ = torch.cuda.mem_get_info(dev)
    L = w.L
    per_spin = 8 if w.model == workloads.ISING else 4
    while L > 64 and L * L // per_spin > free - (2 << 30):
        L //= 2
    return L


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=16)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="ising_L2p20", choices=sorted(workloads.CONFIGS))
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--scheme", type=int, default=1)
    ap.add_argument("--L", type=int, default=0, help="override the lattice side (debugging)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--measure-rmax", type=int, default=-1,
                    help="r_max of the separately timed measurement pass (-1: the workload's)")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: ONE lattice in row slabs over the ranks (strong scaling, fused halo "
                         "mirroring over peer memory) instead of independent replicas")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"])
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.sharded:
        return run_sharded(args)

    import torch
    import torch.distributed as dist
    import paper_2503_14688_b200 as lat
    from paper_2503_14688_b200 import replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    local %= max(torch.cuda.device_count(), 1)     # more ranks than GPUs only in tests (gloo)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        if args.dist_backend == "nccl":
            dist.init_process_group("nccl", device_id=dev)
        else:
            dist.init_process_group("gloo")

    w = workloads.CONFIGS[args.workload]
    L = args.L or pick_L(w, torch, dev)
    cdev = dev if args.dist_backend == "nccl" else "cpu"   # where the plumbing tensors live
    L = replicas.agree_min(L, cdev)             # all replicas use the same size
    g = lat.Lattice(L, w.model, w.delta, seed=replicas.replica_seed(w.seed, rank), scheme=args.scheme,
                    device=str(dev))
    updates_per_step = L * L

    def barrier():
        replicas.barrier()
        torch.cuda.synchronize(dev)

    def timed(fn, steps, start_t):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record(g.stream)
        for k in range(steps):
            fn(start_t + k)
        ev1.record(g.stream)
        torch.cuda.synchronize(dev)
        ms = replicas.max_over_ranks(ev0.elapsed_time(ev1), cdev)
        barrier()
        return ms

    sched = w.beta_schedule(2 * (args.warmup + args.steps) + 16)

    def step_device(t):
        g.sweep(sched[t:t + 1])

    e2e_out = {}

    def step_e2e(t):
        g.sweep(sched[t:t + 1])                 # host fp64 beta in
        e2e_out["r"] = g.measure(1)             # host int64 counts out (synchronises)

    # ---- device-resident timing ------------------------------------------------------------
    for k in range(args.warmup):
        step_device(k)
    n0 = g.launches
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms = timed(step_device, args.steps, args.warmup)
    clocks = sampler.stop() if rank == 0 else {}
    launches = g.launches - n0
    tdone = args.warmup + args.steps

    # ---- end-to-end timing (host buffers in and out every step) ------------------------------
    step_e2e(tdone)
    e2e_ms = timed(step_e2e, args.steps, tdone + 1)
    tdone += 1 + args.steps

    # ---- measurement pass, timed separately --------------------------------------------------
    r_meas = w.r_max if args.measure_rmax < 0 else args.measure_rmax
    r_meas = max(1, min(r_meas, L // 2))
    meas = None
    if rank == 0:
        # ~3e12 (word, r) pairs/s per axis (profiles/): bound the default run to a few seconds
        words = L * L // 32
        if args.measure_rmax < 0 and words * r_meas > 1 << 42:     # an explicit --measure-rmax is honoured
            r_meas = max(1, (1 << 42) // words)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(g.stream)
        M, Q, Sx, Sy = g.measure(r_meas)
        ev1.record(g.stream)
        torch.cuda.synchronize(dev)
        xi_v, r_cut = lat.xi(Sx, Sy, Q, L)
        meas = {"r_max": r_meas, "ms": ev0.elapsed_time(ev1), "t": g.time, "M": M,
                "e": lat.energy(Sx, Sy, Q, w.delta, L), "xi": xi_v, "r_cut": r_cut}
    # ---- worst-case input: the all-up state (every site has 4 aligned neighbours, so every
    # lane needs a random decision and ties are ~3x more frequent than after the quench) ----------
    worst = None
    if world == 1:
        g.fill(1)
        nw = max(2, min(4, args.steps))
        g.sweep(sched[tdone:tdone + 1])
        worst_ms = timed(step_device, nw, tdone + 1)
        tdone += 1 + nw
        worst = {"value": updates_per_step * nw / (worst_ms * 1e6), "unit": UNIT, "steps": nw,
                 "input": "all spins up at t0 (SURVEY.md 8(d) worst case), then the same sweeps"}

    barrier()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = replicas.job_rate(updates_per_step * args.steps, world, ms)
    e2e_value = replicas.job_rate(updates_per_step * args.steps, world, e2e_ms)
    peak, peak_src, sm_max = measured_peaks()
    bpu = BYTES_PER_UPDATE[w.model]
    launch_ms = ms / max(launches, 1)
    alg_bytes = bpu * updates_per_step / 2          # per half-sweep launch
    achieved = alg_bytes / (launch_ms * 1e-3) / 1e9
    in_l2 = lat.state_bytes(L, w.model) <= (126 << 20)
    roofline_hbm = {"bound": "hbm", "kernel": KERNEL[w.model], "achieved": achieved, "peak": peak,
                    "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                    "bytes_per_update": bpu, "launch_ms": launch_ms, "l2_resident": in_l2}
    # the binding roofline: the 16-lane integer dispatch (ALU pipe + IMAD.WIDE), DESIGN.md section 6
    mhz = clocks.get("sm_mhz") or sm_max
    ipu, ipu_exe = ALG_HALF_RATE_INSTR_PER_UPDATE[w.model], EXE_HALF_RATE_INSTR_PER_UPDATE[w.model]
    peak_alu = SM_COUNT * HALF_RATE_LANES_PER_CLK_PER_SM * mhz * 1e6 / 1e12
    ach_alu = ipu * (updates_per_step / 2) / (launch_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": KERNEL[w.model], "achieved": ach_alu, "peak": peak_alu,
                "unit": "T thread-instr/s", "frac": ach_alu / peak_alu,
                "traffic": DRAM_BYTES_PER_UPDATE_NCU[w.model] * updates_per_step / 2,
                "traffic_source": "ncu dram bytes per update (profiles/) x updates per launch",
                "instr_per_update": ipu, "executed_instr_per_update": ipu_exe,
                "executed_frac": ach_alu / peak_alu * ipu_exe / ipu,
                "sm_mhz": mhz, "launch_ms": launch_ms,
                "peak_source": "148 SM x 64 lanes/clk (ALU + IMAD.WIDE dispatch) x sampled SM clock",
                "hbm_frac": achieved / peak, "hbm_achieved_GBs": achieved, "hbm_peak_GBs": peak}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": w.name if L == w.L else f"{w.name}@L={L}", "model": ["ising", "blume-capel"][w.model],
                   "L": L, "spins": L * L, "state_bytes": lat.state_bytes(L, w.model),
                   "beta": float(sched[0]), "rng_scheme": args.scheme, "seed": w.seed,
                   "l2": "inputs_larger_than_l2" if not in_l2 else "l2_resident_by_design",
                   "parallelism": "replicas" if world > 1 else "single"},
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8,
                "d2h_bytes_per_step": 8 * (2 + 4 * 1), "ms_per_step": e2e_ms / args.steps,
                "what": "lattice_sweep(1, host beta) + lattice_measure(r_max=1) -> host int64"},
        "roofline": roofline,
        "roofline_hbm": roofline_hbm,
        "worst_case": worst,
        "measure": meas,
    }
    if not args.no_cpu_baseline:
        Ls, ns = min(L, 4096), 96
        rate, dt, cores = oracle_rate(w, Ls, ns, args.scheme)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{ns} sweeps of a {Ls}x{Ls} lattice of the same model, "
                                          f"beta and RNG scheme ({dt:.1f} s)"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
