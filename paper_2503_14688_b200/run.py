"""Run one workload end to end and write its measurement records as JSON lines.

    python -m paper_2503_14688_b200.run --workload ising_L4096 [--sweeps N] [--r-max R]
                                        [--out records.jsonl] [--checkpoint state.npz]

A record is written at sweeps {0} u {2^k <= N} u {N} (reading 2) and holds the exact
integer counts M, Q, S_x(r), S_y(r) verbatim plus the derived fp64 numbers e, m, q, xi
(Eq. 2-3 and C1 of the paper; readings 8, 10, 14).  Everything on the device runs in
the CUDA kernels behind the C ABI; this script only drives it.

--checkpoint writes (packed words, sweep counter, seed, model, delta, scheme) after the last
sweep; --resume continues from such a file.  Because the random numbers are counter-based
(keyed by seed, sweep, colour, site), a resumed run is bit-identical to an uninterrupted one.
"""
from __future__ import annotations

import argparse
import json
import sys
import time

import numpy as np

from . import binding as lat
from . import workloads


def record(g: "lat.Lattice", r_max: int, delta: float) -> dict:
    M, Q, Sx, Sy = g.measure(r_max)
    L = g.L
    xi, r_cut = lat.xi(Sx, Sy, Q, L)
    n = float(L) * float(L)
    return {"t": g.time, "L": L, "M": M, "Q": Q, "Sx": Sx.tolist(), "Sy": Sy.tolist(),
            "e": lat.energy(Sx, Sy, Q, delta, L), "m": M / n, "q": Q / n, "xi": xi, "r_cut": r_cut}


def save_checkpoint(g: "lat.Lattice", path: str) -> None:
    g.synchronize()
    np.savez(path, words=g.buf.cpu().numpy(), t=g.time, seed=np.uint64(g.seed), model=g.model,
             delta=g.delta, scheme=g.scheme, L=g.L)


def load_checkpoint(path: str, device: str = "cuda:0") -> "lat.Lattice":
    import torch
    z = np.load(path)
    g = lat.Lattice(int(z["L"]), int(z["model"]), float(z["delta"]), int(z["seed"]), int(z["scheme"]),
                    device=device)
    g.buf.copy_(torch.from_numpy(z["words"]).to(g.buf.device))
    g.set_time(int(z["t"]))
    return g


def run(w: workloads.Workload, sweeps: int | None = None, r_max: int | None = None, out=None,
        L: int | None = None, resume: str | None = None, device: str = "cuda:0") -> list[dict]:
    """Run `sweeps` sweeps of workload w (optionally on a smaller lattice L), recording at 2^k."""
    sweeps = w.sweeps if sweeps is None else sweeps
    if resume:
        g = load_checkpoint(resume, device)
    else:
        g = lat.Lattice(L or w.L, w.model, w.delta, w.seed, device=device)
    r_max = min(w.r_max if r_max is None else r_max, g.L // 2)
    records = []
    for t in w.measure_times(sweeps):
        if t < g.time:
            continue
        if t > g.time:
            t0 = time.perf_counter()
            g.sweep(w.beta_schedule(t - g.time, g.time))
            g.synchronize()
            dt = time.perf_counter() - t0
        else:
            dt = 0.0
        rec = record(g, r_max, w.delta)
        rec["workload"], rec["seconds_since_last_record"] = w.name, dt
        records.append(rec)
        if out is not None:
            out.write(json.dumps(rec) + "\n")
            out.flush()
    run.last_lattice = g
    return records


def replica_correlations(w: workloads.Workload, n_runs: int, sweeps: int, r_max: int, L: int | None = None,
                         device: str = "cuda:0", batch: int | None = None):
    """n_runs independent realisations of workload w (seeds w.seed + 7919 k): returns
    (times[T], C[T][run, r] for r = 0..r_max, e[T][run]) at the record times 2^k <= sweeps --
    the input of the estimator layer (analysis.py).  The realisations run as batches of replicas
    (lattice_create_batch): `batch` per handle, by default as many as fit in 1/4 of the free
    device memory, so that small lattices fill the GPU."""
    import torch
    from . import analysis
    L = L or w.L
    times = [t for t in w.measure_times(sweeps) if t > 0]
    C = [np.zeros((n_runs, r_max + 1)) for _ in times]
    e = [np.zeros(n_runs) for _ in times]
    if batch is None:
        free, _ = torch.cuda.mem_get_info(torch.device(device))
        batch = max(1, min(n_runs, (free // 4) // lat.state_bytes(L, w.model)))
    for k0 in range(0, n_runs, batch):
        nb = min(batch, n_runs - k0)
        seeds = np.array([w.seed + 7919 * (k0 + k) for k in range(nb)], dtype=np.uint64)
        g = lat.LatticeBatch(L, seeds, w.model, w.delta, device=device)
        for a, t in enumerate(times):
            g.sweep(w.beta_schedule(t - g.time, g.time))
            M, Q, Sx, Sy = g.measure(r_max)
            for k in range(nb):
                C[a][k0 + k] = analysis.correlation(Sx[k], Sy[k], L, Q[k])
                e[a][k0 + k] = lat.energy(Sx[k], Sy[k], Q[k], w.delta, L)
        g.close()
    return np.array(times, dtype=np.float64), C, e


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--workload", required=True, choices=sorted(workloads.CONFIGS))
    ap.add_argument("--sweeps", type=int, default=None)
    ap.add_argument("--r-max", type=int, default=None)
    ap.add_argument("--L", type=int, default=None, help="run the workload's recipe on a smaller lattice")
    ap.add_argument("--out", default="-")
    ap.add_argument("--checkpoint", default=None)
    ap.add_argument("--resume", default=None)
    a = ap.parse_args(argv)
    w = workloads.CONFIGS[a.workload]
    out = sys.stdout if a.out == "-" else open(a.out, "w")
    run(w, a.sweeps, a.r_max, out, a.L, a.resume)
    if a.checkpoint:
        save_checkpoint(run.last_lattice, a.checkpoint)
    if out is not sys.stdout:
        out.close()
    return 0


if __name__ == "__main__":
    raise SystemExit(main())

