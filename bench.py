#!/usr/bin/env python
"""bench.py -- spin updates/ns of the checkerboard Metropolis sweep on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

A "step" is one full-lattice Metropolis sweep (black half-sweep + white half-sweep, thresholds
rebuilt from the step's beta on the host) of BASELINE.json's throughput configuration:
2D Ising, L = 2^20 (128 GiB at 1 bit/spin), disordered start, beta_c.  If the device cannot
hold 128 GiB the largest power-of-two L that fits is used and named in config.workload.  For
workloads whose sweep takes less than ~2 s / K a step is `sweeps_per_step` sweeps issued as ONE
lattice_sweep(n) call (the persistent multi-sweep path where it applies), chosen so that the K
timed steps last at least --min-seconds (default 2 s): every quoted number then has clock
samples (config.sweeps_per_step says how many).

One JSON line is printed by rank 0:
  value     whole-job spin updates/ns, device-timed (CUDA events), lattice resident in HBM
  e2e       the same metric through the C-ABI with host buffers every step: the step's beta goes
            in as a host fp64 array and the step's result (M, Q, S_x(1), S_y(1) -> e, m) comes
            back to host memory (lattice_sweep_record), all inside the timed region
  roofline  the binding roofline of the dominant kernel (the half-sweep): "bound": "alu" --
            ALGORITHMIC thread-instructions of the half-rate dispatch class per launch (hand
            count) / mean launch time measured here, against a peak MEASURED
            in this run: lattice_ubench_int_dispatch lanes/clk/SM x SMs x the sampled SM clock.
            `executed_frac` and `traffic` use constants from the committed ncu capture named in
            `profile` (not from this run; `stale_profile` says whether the kernel sources changed
            since that capture)
  roofline_hbm  the HBM roofline BASELINE.json's metric asks for: algorithmic bytes (0.375
            B/update Ising, 0.75 BC: read both colours once, write one) / mean launch time,
            against the measured copy bandwidth in MEASURED_PEAKS.json
  blume_capel   (default invocation, 1 GPU) the same measurements for Blume-Capel at the paper's
            size (L = 2^19) and for BASELINE config 5b (L = 2^15, beta ramp), each
            with its own value, e2e, roofline, roofline_hbm and clocks
  batched_replicas  (default invocation, 1 GPU) aggregate updates/ns of 64 replicas of L = 4096 and
            8192 replicas of L = 64 in one batch handle each (lattice_create_batch): the shapes of
            BASELINE configs 2 and 1, which fill the GPU only as batches
  cpu_baseline  the oracle, as it stands, on the host cores over bounded samples: `value` is the
            all-cores figure for the timed model and RNG scheme; `matrix` holds 1 thread and all
            cores x schemes 0/1 x both models, `cpu_model` the CPU
  measure   the measurement pass (M, Q, C(r) on both axes) timed separately after the sweeps; on the
            tensor-core path with its own `roofline` ("bound": "tensor"): band-Gram flops / time against
            2 x the measured sustained bf16 peak (fp8 operands)

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
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2503_14688_b200 import profile_constants as pc  # noqa: E402
from paper_2503_14688_b200 import workloads  # noqa: E402

METRIC = "spin updates/ns per B200 (Ising & Blume-Capel) and % of HBM roofline"
UNIT = "spin updates/ns"
KERNEL = {workloads.ISING: "ising_march_kernel", workloads.BLUME_CAPEL: "bc_march_kernel"}
MODEL_NAME = ["ising", "blume-capel"]


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(p.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


class ClockSampler:
    """SM clock and throttle reasons of one GPU during a timed region.

    In-process through NVML (pynvml): one sample when the region starts, one every 20 ms from a
    thread, one when it ends -- so even a region of a few milliseconds has >= 2 samples.  If
    NVML cannot be loaded the profiling recipe's `nvidia-smi -lms` line is used instead."""
    BAD = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
           0x80: "hw_power_brake_slowdown"}
    NOTE = {0x4: "sw_power_cap"}
    SMI_FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
                  "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                  "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, torch, dev):
        self.nv, self.h, self.index = None, None, dev.index or 0
        self.sm, self.reasons, self.power = [], set(), []
        self.sm_max = None
        self._stop, self._thr, self._smi, self._smi_path = threading.Event(), None, None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            uuid = getattr(torch.cuda.get_device_properties(dev), "uuid", None)
            h = None
            if uuid is not None:
                for cand in (f"GPU-{uuid}", str(uuid)):
                    try:
                        h = pynvml.nvmlDeviceGetHandleByUUID(cand.encode() if isinstance(cand, str) else cand)
                        break
                    except Exception:
                        h = None
            if h is None:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
                ids = [v for v in vis.split(",") if v.strip().isdigit()]
                phys = int(ids[self.index]) if self.index < len(ids) else self.index
                h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.nv, self.h = pynvml, h
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _sample(self):
        nv = self.nv
        try:
            self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
            try:
                mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
            except Exception:
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            for bit, name in {**self.BAD, **self.NOTE}.items():
                if mask & bit:
                    self.reasons.add(name)
            self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
        except Exception:
            pass

    def _loop(self):
        while not self._stop.wait(0.02):
            self._sample()

    def start(self):
        self.sm, self.reasons, self.power = [], set(), []
        self._stop.clear()
        if self.nv is not None:
            self._sample()
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
            return
        try:
            fd, self._smi_path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self._smi = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.SMI_FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=open(self._smi_path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self._smi = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": 0, "source": "none"}
        if self.nv is not None:
            self._stop.set()
            if self._thr is not None:
                self._thr.join(timeout=2)
            self._sample()
            out["source"] = "nvml in-process, 20 ms"
        elif self._smi is not None:
            self._smi.terminate()
            try:
                self._smi.wait(timeout=5)
            except Exception:
                self._smi.kill()
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            mx = []
            try:
                for line in open(self._smi_path):
                    f = [x.strip() for x in line.split(",")]
                    if len(f) < 9:
                        continue
                    try:
                        self.sm.append(float(f[1])); mx.append(float(f[2]))
                    except ValueError:
                        continue
                    for name, v in zip(names, f[5:9]):
                        if v.lower().startswith("active"):
                            self.reasons.add(name)
                os.unlink(self._smi_path)
            except Exception:
                pass
            if mx:
                out["sm_max_mhz"] = float(max(mx))
            out["source"] = "nvidia-smi -lms 100"
        if self.sm:
            out.update(sm_mhz=float(np.median(self.sm)), sm_min_mhz=float(min(self.sm)), samples=len(self.sm))
        if self.power:
            out["power_w_max"] = float(max(self.power))
        out["reasons"] = sorted(self.reasons)
        return out


def oracle_rate(model, delta, seed, beta, L, sweeps, scheme=1, threads=None):
    """Updates/ns of the CPU oracle on `sweeps` sweeps of an L x L sample; (rate, seconds, threads)."""
    import oracle
    oracle.build()
    oracle.set_threads(threads or os.cpu_count() or 1)
    used = oracle.get_threads()
    o = oracle.OracleLattice(L, model, delta, seed, scheme)
    b = np.full(sweeps, beta, dtype=np.float64)
    t0 = time.perf_counter()
    o.sweep(b)
    dt = time.perf_counter() - t0
    o.close()
    return L * L * sweeps / dt / 1e9, dt, used


def cpu_baseline_matrix(w, scheme):
    """BASELINE.md section 3 / SURVEY.md section 8(d): the oracle as it stands, 1 thread and all host cores,
    RNG schemes 0 and 1, both models, on bounded samples (~2 s each, ~20 s in total)."""
    cores = os.cpu_count() or 1
    rows = []
    for model, delta, beta in ((workloads.ISING, 0.0, workloads.BETA_C_ISING),
                               (workloads.BLUME_CAPEL, 0.0, workloads.BETA_BC)):
        for sch in (0, 1):
            for thr, L, ns in ((1, 1024, 8), (cores, 4096, 8)):
                rate, dt, used = oracle_rate(model, delta, w.seed, beta, L, ns, sch, thr)
                rows.append({"model": MODEL_NAME[model], "rng_scheme": sch, "threads": used, "value": rate,
                             "unit": UNIT, "sample": f"{ns} sweeps of {L}x{L}", "seconds": round(dt, 2)})
    beta0 = float(w.beta_schedule(1)[0])
    Ls, ns = min(w.L, 4096), 48
    rate, dt, used = oracle_rate(w.model, w.delta, w.seed, beta0, Ls, ns, scheme, cores)
    return {"value": rate, "unit": UNIT, "cores": used, "kind": "oracle", "cpu_model": cpu_model(),
            "sample": f"{ns} sweeps of a {Ls}x{Ls} lattice of the timed model ({MODEL_NAME[w.model]}), "
                      f"beta and RNG scheme {scheme} ({dt:.1f} s); matrix: 8 sweeps of 1024^2 (1 thread) / "
                      f"4096^2 (all cores)",
            "matrix": rows}


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, same metric and config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workloads.CONFIGS[args.workload]
    Ls, ns = min(w.L, 4096), 8                   # one step = 8 sweeps of a 4096 x 4096 sample (~1 s)
    beta0 = float(w.beta_schedule(1)[0])
    for _ in range(args.warmup):
        oracle_rate(w.model, w.delta, w.seed, beta0, 256, 1)
    t0 = time.perf_counter()
    rates = [oracle_rate(w.model, w.delta, w.seed, beta0, Ls, ns) for _ in range(args.steps)]
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
                         "kind": "oracle", "sample": sample, "cpu_model": cpu_model()},
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


_UBENCH = {}


def dispatch_peak(lat, torch, dev, stream_ptr):
    """Measured integer-dispatch rates (thread-instr/clk/SM) from the library's micro-benchmark,
    once per process: {"lop3", "mulwide_lop3", "mulwide_3lop3", "popc"}."""
    if not _UBENCH:
        with torch.cuda.device(dev):
            for mode, name in enumerate(("lop3", "mulwide_lop3", "mulwide_3lop3", "popc")):
                v, _ = lat.binding.ubench_int_dispatch(mode, stream_ptr)
                _UBENCH[name] = v
    return dict(_UBENCH)


def bench_workload(w, args, lat, torch, dev, rank, world, cdev, replicas, *, measure_pass, worst_case):
    """Time workload w (device-resident and end to end); returns the pieces of the JSON line."""
    L = args.L or pick_L(w, torch, dev)
    L = replicas.agree_min(L, cdev)             # all replicas use the same size
    g = lat.Lattice(L, w.model, w.delta, seed=replicas.replica_seed(w.seed, rank), scheme=args.scheme,
                    device=str(dev))
    if args.no_persistent:
        g.set_persist_blocks(0xffffffff)
    if args.force_persistent:
        g.set_persist_blocks(1 << 20)
    updates_per_sweep = L * L
    K, W = args.steps, args.warmup

    def barrier():
        replicas.barrier()
        torch.cuda.synchronize(dev)

    def timed(fn, steps, start_t, sps):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record(g.stream)
        for k in range(steps):
            fn(start_t + k * sps, sps)
        ev1.record(g.stream)
        torch.cuda.synchronize(dev)
        ms = replicas.max_over_ranks(ev0.elapsed_time(ev1), cdev)
        barrier()
        return ms

    def sched(t, n):
        return w.beta_schedule(n, t)

    def step_device(t, n):
        g.sweep(sched(t, n))

    e2e_out = {}

    def step_e2e(t, n):
        # host fp64 beta in, host int64 counts out (synchronises): one C-ABI call, lattice_sweep_record
        e2e_out["r"] = g.sweep_record(sched(t, n))

    peaks = dispatch_peak(lat, torch, dev, g.stream.cuda_stream)

    # ---- warm-up (W steps of one sweep), then size the step so that K steps last >= min_seconds ----
    t_now = 0
    for _ in range(max(W - 1, 0)):
        step_device(t_now, 1)
        t_now += 1
    est_ms = timed(step_device, 1, t_now, 1) if W >= 1 else 1.0
    t_now += 1 if W >= 1 else 0
    sps = 1
    if args.min_seconds > 0 and K * est_ms < args.min_seconds * 1e3:
        want_ms = args.min_seconds * 1e3 / K
        sps = int(min(max(1, np.ceil(want_ms / max(est_ms, 1e-3))), 65536))
        # second calibration at the real step size: several sweeps per call run faster than one
        # (persistent kernel, no launch gaps), so the first guess is usually too small
        for _ in range(2):
            ms1 = timed(step_device, 1, t_now, sps)
            t_now += sps
            if ms1 >= want_ms or sps >= 65536:
                break
            sps = int(min(np.ceil(sps * want_ms / max(ms1, 1e-3) * 1.05), 65536))
        sps = -int(replicas.agree_min(-sps, cdev)) if world > 1 else sps     # the largest over ranks
        step_device(t_now, sps)                 # one untimed step of the final size
        t_now += sps

    # ---- device-resident timing ------------------------------------------------------------
    n0 = g.launches
    sampler = ClockSampler(torch, dev)
    if rank == 0:
        sampler.start()
    ms = timed(step_device, K, t_now, sps)
    clocks = sampler.stop() if rank == 0 else {}
    launches = g.launches - n0
    t_now += K * sps

    # ---- end-to-end timing (host buffers in and out every step) ------------------------------
    step_e2e(t_now, sps)
    t_now += sps
    if rank == 0:
        sampler.start()
    e2e_ms = timed(step_e2e, K, t_now, sps)
    e2e_clocks = sampler.stop() if rank == 0 else {}
    t_now += K * sps

    # ---- measurement pass, timed separately --------------------------------------------------
    meas = None
    if measure_pass and rank == 0:
        r_meas = w.r_max if args.measure_rmax < 0 else args.measure_rmax
        r_meas = max(1, min(r_meas, L // 2))
        # the tensor-core path (csrc/corr_tc2.cuh) does C(r <= 4096) at L = 2^20 in ~8 s: the default run
        # measures the workload's full r_max; only where that path does not apply (L < 4096) and the
        # XOR/popcount kernels would take long is r_max bounded (an explicit --measure-rmax is honoured)
        words = L * L // 32
        if args.measure_rmax < 0 and L < 4096 and words * r_meas > 1 << 42:
            r_meas = max(1, (1 << 42) // words)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(g.stream)
        M, Q, Sx, Sy = g.measure(r_meas)
        ev1.record(g.stream)
        torch.cuda.synchronize(dev)
        xi_v, r_cut = lat.xi(Sx, Sy, Q, L)
        sparse = None
        if args.measure_list > 0:
            # the paper's sparse sampling in r: log-spaced separations up to r_meas
            rl = sorted({max(1, int(round(r_meas ** (k / max(args.measure_list - 1, 1))))) for k in range(args.measure_list)})
            ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev2.record(g.stream)
            Ml, Ql, Sxl, Syl = g.measure_list(rl)
            ev3.record(g.stream)
            torch.cuda.synchronize(dev)
            same = all(int(Sxl[k]) == int(Sx[r - 1]) and int(Syl[k]) == int(Sy[r - 1]) for k, r in enumerate(rl))
            sparse = {"points": len(rl), "r_last": rl[-1], "ms": ev2.elapsed_time(ev3), "equals_dense": bool(same and Ml == M)}
        tc_roofline = None
        if L >= 4096 and r_meas >= 48:
            # dense C(r) as the band of the row / column Gram matrix (csrc/corr_tc2.cuh): per axis L / 256 pair
            # tiles x ceil((r_max + 256) / 512) passes of 256 x 512 outputs, contraction length L
            passes = (r_meas + 256 + 511) // 512
            flop = 2.0 * 2 * (L // 256) * passes * 256 * 512 * L
            tf = flop / (ev0.elapsed_time(ev1) * 1e-3) / 1e12
            try:
                with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
                    mp = json.load(f)
                bf16 = float(mp.get("bf16_tflops_sustained") or mp["bf16_tflops"])
                src = "2 x the sustained bf16 TFLOP/s of MEASURED_PEAKS.json (the guide's nominal fp8 : bf16 ratio)"
            except Exception:
                bf16, src = 2250.0, "2 x the nominal 2250 bf16 TFLOP/s (no MEASURED_PEAKS.json)"
            tc_roofline = {"bound": "tensor", "kernel": "corr_tc2_kernel (+ band_transpose_kernel, measure_mq_kernel)",
                           "achieved": tf, "peak": 2.0 * bf16, "unit": "TFLOP/s", "frac": tf / (2.0 * bf16),
                           "dtype": "fp8 e4m3 operands, fp32 accumulate (exact integers)", "peak_source": src,
                           "flop": flop, "traffic": None}
        meas = {"r_max": r_meas, "ms": ev0.elapsed_time(ev1), "t": g.time, "M": M, "roofline": tc_roofline,
                "path": "tensor cores (tcgen05 banded Gram: CTA pairs, x axis on transposed bands; csrc/corr_tc2.cuh, corr_transpose.cuh)" if (L >= 4096 and r_meas >= 48)
                        else "XOR/popcount kernels (csrc/measure.cuh)",
                "e": lat.energy(Sx, Sy, Q, w.delta, L), "xi": xi_v, "r_cut": r_cut, "sparse_list": sparse}
    # ---- worst-case input: the all-up state (every site has 4 aligned neighbours, so every
    # lane needs a random decision and ties are ~3x more frequent than after the quench) ----------
    worst = None
    if worst_case and world == 1:
        g.fill(1)
        nw = max(2, min(4, K))
        step_device(t_now, sps)
        t_now += sps
        worst_ms = timed(step_device, nw, t_now, sps)
        t_now += nw * sps
        worst = {"value": updates_per_sweep * nw * sps / (worst_ms * 1e6), "unit": UNIT, "steps": nw,
                 "input": "all spins up at t0 (SURVEY.md 8(d) worst case), then the same sweeps"}
    barrier()
    state_bytes = lat.state_bytes(L, w.model)
    g.close()
    del g
    torch.cuda.empty_cache()

    # ---- rooflines ---------------------------------------------------------------------------
    updates = updates_per_sweep * sps * K
    value = replicas.job_rate(updates, world, ms)
    e2e_value = replicas.job_rate(updates, world, e2e_ms)
    peak, peak_src, sm_max = measured_peaks()
    cap = pc.captured(w.model)
    bpu = pc.ALGORITHMIC_BYTES_PER_UPDATE[w.model]
    half_sweeps = 2 * sps * K
    hs_ms = ms / half_sweeps                    # mean duration of one half-sweep (one launch, or one
    upl = updates_per_sweep / 2                 # colour pass inside the persistent kernel)
    achieved = bpu * upl / (hs_ms * 1e-3) / 1e9
    in_l2 = state_bytes <= (126 << 20)
    roofline_hbm = {"bound": "hbm", "kernel": KERNEL[w.model], "achieved": achieved, "peak": peak,
                    "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                    "bytes_per_update": bpu, "half_sweep_ms": hs_ms, "l2_resident": in_l2}
    mhz = clocks.get("sm_mhz") or sm_max
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    lanes = peaks["mulwide_3lop3"]
    ipu = pc.ALGORITHMIC_HALF_RATE_INSTR_PER_UPDATE[w.model]
    ipu_exe = cap["executed_half_rate_instr_per_update"]
    peak_alu = sms * lanes * mhz * 1e6 / 1e12
    ach_alu = ipu * upl / (hs_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": KERNEL[w.model], "achieved": ach_alu, "peak": peak_alu,
                "unit": "T thread-instr/s", "frac": ach_alu / peak_alu,
                "frac_is": "model: algorithmic instruction count (DESIGN.md section 6) x updates / launch time "
                           "measured in this run, over the dispatch peak measured in this run",
                "traffic": cap["dram_bytes_per_update"] * upl,
                "traffic_source": f"constant from {cap['profile']} (ncu dram__bytes_read+write per update at commit "
                                  f"{cap['commit']}) x updates per launch; NOT measured in this run",
                "instr_per_update_algorithmic": ipu,
                "instr_per_update_executed": ipu_exe,
                "executed_source": f"constant from {cap['profile']} (commit {cap['commit']}); not this run",
                "executed_frac": ach_alu / peak_alu * ipu_exe / ipu,
                "stale_profile": cap["stale_profile"],
                "sm_mhz": mhz, "half_sweep_ms": hs_ms,
                "peak_lanes_per_clk_per_sm": lanes, "sm_count": sms,
                "peak_source": "measured in this run: lattice_ubench_int_dispatch (1 mul.wide.u32 + 3 LOP3 chains, "
                               "clock64) x SM count x sampled SM clock",
                "ubench_thread_instr_per_clk_per_sm": peaks,
                "hbm_frac": achieved / peak, "hbm_achieved_GBs": achieved, "hbm_peak_GBs": peak}
    return {
        "value": value, "ms_per_step": ms / K, "L": L,
        "config": {"workload": w.name if L == w.L else f"{w.name}@L={L}", "model": MODEL_NAME[w.model],
                   "L": L, "spins": L * L, "state_bytes": state_bytes,
                   "beta": float(w.beta_schedule(1)[0]), "rng_scheme": args.scheme, "seed": w.seed,
                   "sweeps_per_step": sps, "timed_seconds": ms / 1e3, "persistent_kernel_allowed": not args.no_persistent,
                   "l2": "inputs_larger_than_l2" if not in_l2 else "l2_resident_by_design",
                   "parallelism": "replicas" if world > 1 else "single"},
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * sps,
                "d2h_bytes_per_step": 8 * (2 + 4 * 1), "ms_per_step": e2e_ms / K, "clocks": e2e_clocks,
                "what": f"lattice_sweep_record({sps}, host beta[{sps}]) -> host int64 (M, Q, S_x(1), S_y(1)), per step: the "
                        f"sweeps and the r = 1 record (fused into the last white half-sweep for Ising marching lattices, "
                        f"else lattice_sweep + lattice_measure(1))"},
        "roofline": roofline, "roofline_hbm": roofline_hbm, "worst_case": worst, "measure": meas,
    }


def bench_batch(name, L, n_rep, args, lat, torch, dev):
    """Aggregate updates/ns of n_rep independent Ising replicas of side L in one batch handle
    (lattice_create_batch) at beta_c: K steps of `sps` sweeps per lattice_sweep call, sized to
    --min-seconds, clock-sampled; e2e adds lattice_measure_batch(r_max = 1) per step."""
    seeds = np.arange(n_rep, dtype=np.uint64) * 1000 + np.uint64(workloads.SEED_BASE + 31)
    b = lat.LatticeBatch(L, seeds, lat.ISING, 0.0, args.scheme, device=str(dev))
    if args.no_persistent:                          # A/B: two launches per sweep instead of the in-kernel sweep loops
        lat.lib().lattice_set_persist_blocks(b._h, 0xffffffff)
    K = args.steps
    beta = workloads.BETA_C_ISING

    def timed(fn, steps, sps):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        ev0.record(b.stream)
        for _ in range(steps):
            fn(sps)
        ev1.record(b.stream)
        torch.cuda.synchronize(dev)
        return ev0.elapsed_time(ev1)

    def step_device(n):
        b.sweep(np.full(n, beta))

    def step_e2e(n):
        b.sweep(np.full(n, beta))
        b.measure(1)

    for _ in range(max(args.warmup, 1)):
        step_device(4)
    sps, want_ms = 4, args.min_seconds * 1e3 / K
    for _ in range(3):
        ms1 = timed(step_device, 1, sps)
        if ms1 >= want_ms or sps >= 65536:
            break
        sps = int(min(np.ceil(sps * want_ms / max(ms1, 1e-3) * 1.05), 65536))
    n0 = b.launches
    sampler = ClockSampler(torch, dev)
    sampler.start()
    ms = timed(step_device, K, sps)
    clocks = sampler.stop()
    launches = b.launches - n0
    step_e2e(sps)
    sampler.start()
    e2e_ms = timed(step_e2e, K, sps)
    e2e_clocks = sampler.stop()
    b.close()
    del b
    torch.cuda.empty_cache()
    updates = L * L * n_rep * sps * K
    return {"value": updates / (ms * 1e6), "unit": UNIT, "steps": K, "ms_per_step": ms / K,
            "config": {"workload": name, "model": "ising", "L": L, "replicas": n_rep, "spins": L * L * n_rep,
                       "state_bytes": L * L // 8 * n_rep, "beta": beta, "rng_scheme": args.scheme,
                       "sweeps_per_step": sps, "timed_seconds": ms / 1e3,
                       "l2": "l2_resident_by_design" if L * L // 8 * n_rep <= (126 << 20) else "inputs_larger_than_l2"},
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": updates / (e2e_ms * 1e6), "unit": UNIT, "h2d_bytes_per_step": 8 * sps,
                    "d2h_bytes_per_step": 8 * 6 * n_rep, "ms_per_step": e2e_ms / K, "clocks": e2e_clocks,
                    "what": f"lattice_sweep({sps}) on the batch + lattice_measure_batch(r_max=1) -> host int64 per replica"}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=16)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="ising_L2p20", choices=sorted(workloads.CONFIGS))
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--scheme", type=int, default=1)
    ap.add_argument("--L", type=int, default=0, help="override the lattice side (debugging)")
    ap.add_argument("--min-seconds", type=float, default=2.0,
                    help="lower bound on the timed region: a step becomes several sweeps per call if needed")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-blume-capel", action="store_true",
                    help="skip the Blume-Capel workloads the default invocation also times")
    ap.add_argument("--no-batches", action="store_true",
                    help="skip the batched-replica workloads the default invocation also times")
    ap.add_argument("--delta", type=float, default=None,
                    help="override the workload's crystal field Delta (Blume-Capel; e.g. the general marching kernel)")
    ap.add_argument("--beta", type=float, default=None, help="override the workload's beta schedule with a constant")
    ap.add_argument("--no-persistent", action="store_true",
                    help="cache-resident lattices: two launches per sweep instead of the persistent multi-sweep kernel (A/B)")
    ap.add_argument("--force-persistent", action="store_true",
                    help="cache-resident lattices: take the persistent multi-sweep kernel wherever it exists (A/B)")
    ap.add_argument("--batches-only", action="store_true",
                    help="time only the batched-replica workloads (profiling aid: prints their JSON object)")
    ap.add_argument("--batch-shapes", default="", help="with --batches-only: LxN[,LxN...] instead of the two default shapes")
    ap.add_argument("--measure-rmax", type=int, default=-1,
                    help="r_max of the separately timed measurement pass (-1: the workload's)")
    ap.add_argument("--measure-list", type=int, default=64,
                    help="also time lattice_measure_list on this many log-spaced separations (0: skip)")
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
    cdev = dev if args.dist_backend == "nccl" else "cpu"   # where the plumbing tensors live

    if args.batches_only:
        shapes = [("ising_L4096_x64", 4096, 64), ("ising_L64_x8192", 64, 8192)]
        if args.batch_shapes:
            shapes = [(f"ising_L{a}_x{b}", int(a), int(b)) for a, b in (x.split("x") for x in args.batch_shapes.split(","))]
        out = {name: bench_batch(name, Lb, nb, args, lat, torch, dev) for name, Lb, nb in shapes}
        print(json.dumps({"batched_replicas": out}))
        return

    w = workloads.CONFIGS[args.workload]
    if args.delta is not None or args.beta is not None:
        import dataclasses
        kw = {}
        if args.delta is not None:
            kw["delta"] = args.delta
        if args.beta is not None:
            kw.update(protocol=1, beta_f=args.beta)
        w = dataclasses.replace(w, name=w.name + "".join(f"@{k}={v}" for k, v in kw.items()), **kw)
    res = bench_workload(w, args, lat, torch, dev, rank, world, cdev, replicas, measure_pass=True, worst_case=True)

    # the metric's second half: Blume-Capel at the paper's size and BASELINE config 5b, same process
    extra = {}
    if world == 1 and not args.no_blume_capel and args.workload == "ising_L2p20" and not args.L:
        for name in ("bc_L2p19", "bc_L2p15_ramp"):
            r = bench_workload(workloads.CONFIGS[name], args, lat, torch, dev, rank, world, cdev, replicas,
                               measure_pass=False, worst_case=True)
            extra[name] = {"value": r["value"], "unit": UNIT, "steps": args.steps, "ms_per_step": r["ms_per_step"],
                           "config": r["config"], "clocks": r["clocks"], "gpu_launches": r["gpu_launches"],
                           "e2e": r["e2e"], "roofline": r["roofline"], "roofline_hbm": r["roofline_hbm"],
                           "worst_case": r["worst_case"]}

    # cache-resident sizes fill the GPU only as batches of replicas (BASELINE configs 1 and 2's shapes)
    batches = {}
    if world == 1 and not args.no_batches and args.workload == "ising_L2p20" and not args.L:
        for name, Lb, nb in (("ising_L4096_x64", 4096, 64), ("ising_L64_x8192", 64, 8192)):
            batches[name] = bench_batch(name, Lb, nb, args, lat, torch, dev)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    line = {
        "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": res["config"], "clocks": res["clocks"], "gpu_launches": res["gpu_launches"],
        "e2e": res["e2e"], "roofline": res["roofline"], "roofline_hbm": res["roofline_hbm"],
        "worst_case": res["worst_case"], "measure": res["measure"],
    }
    if extra:
        line["blume_capel"] = extra
    if batches:
        line["batched_replicas"] = batches
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline_matrix(w, args.scheme)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
