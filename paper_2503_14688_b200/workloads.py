"""Seeded synthetic workloads: the five BASELINE.json configs as plain data.

This module is the only thing the CUDA path's callers (tests, bench.py) and the oracle's
callers share.  It holds no arithmetic of the method: only lattice sizes, seeds, the
temperature schedules handed to `lattice_sweep` as fp64 arrays, and the measurement times.
The paper evaluates on no dataset: every run starts from a seeded fully disordered lattice
(PAPER.md:65), so these configs *are* the workloads.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

ISING, BLUME_CAPEL = 0, 1

#: Onsager: T_c = 2/log(1+sqrt 2), beta_c = log(1+sqrt 2)/2
BETA_C_ISING = math.log(1.0 + math.sqrt(2.0)) / 2.0
#: BASELINE.json config 3: T = 1.6934 (~T_c of Blume-Capel at Delta = 0; PAPER.md:40 has 1.6935583(5))
T_BC = 1.6934
BETA_BC = 1.0 / T_BC

SEED_BASE = 2503146880      # seed = 2503146880 + config index


@dataclass(frozen=True)
class Workload:
    name: str
    model: int
    L: int
    delta: float
    seed: int
    sweeps: int
    r_max: int
    protocol: int = 1                      # 1: constant beta; 2: ramp (BASELINE.json config 5);
                                           # 3: the paper's two-step protocol (Table II)
    beta_f: float = field(default=BETA_C_ISING)
    beta_1: float = 0.0                    # protocol 3: 1/T_1 for sweeps t < t_switch
    t_switch: int = 0

    def beta_schedule(self, n: int | None = None, start: int = 0) -> np.ndarray:
        """beta[t] for sweeps start..start+n-1 as fp64 (what `lattice_sweep` takes)."""
        n = self.sweeps if n is None else n
        t = np.arange(start, start + n, dtype=np.float64)
        if self.protocol == 1:
            return np.full(n, self.beta_f, dtype=np.float64)
        if self.protocol == 3:
            # T_1 until t_switch, then T_2 (beta_f = 1/T_2)
            return np.where(t < float(self.t_switch), self.beta_1, self.beta_f).astype(np.float64)
        # protocol 2: beta ramps linearly from 0.9*beta_f to beta_f over sweeps 0..999
        ramp = 0.9 * self.beta_f + (0.1 * self.beta_f) * (t / 999.0)
        return np.where(t < 999.0, ramp, self.beta_f).astype(np.float64)

    def measure_times(self, n: int | None = None) -> list[int]:
        """Sweep counts after which measurements are recorded: {0} u {2^k <= n} u {n}."""
        n = self.sweeps if n is None else n
        ts = {0, n}
        k = 1
        while k <= n:
            ts.add(k)
            k *= 2
        return sorted(ts)

    @property
    def spins(self) -> int:
        return self.L * self.L

    @property
    def state_bytes(self) -> int:
        return self.L * self.L // (8 if self.model == ISING else 4)


CONFIGS: dict[str, Workload] = {
    # 1: small case the oracle finishes in seconds
    "ising_L64": Workload("ising_L64", ISING, 64, 0.0, SEED_BASE + 1, 2000, 32),
    # 2: cache-resident Ising
    "ising_L4096": Workload("ising_L4096", ISING, 4096, 0.0, SEED_BASE + 2, 20000, 1024),
    # 3: Blume-Capel at Delta = 0, T = 1.6934
    "bc_L16384": Workload("bc_L16384", BLUME_CAPEL, 16384, 0.0, SEED_BASE + 3, 10000, 4096,
                          beta_f=BETA_BC),
    # 4: the throughput run (128 GiB at 1 bit/spin) -- the bench workload
    "ising_L2p20": Workload("ising_L2p20", ISING, 1 << 20, 0.0, SEED_BASE + 4, 64, 4096),
    # 5a/5b: protocol 2 (time-varying beta)
    "ising_L2p16_ramp": Workload("ising_L2p16_ramp", ISING, 1 << 16, 0.0, SEED_BASE + 5, 20000,
                                 1024, protocol=2, beta_f=BETA_C_ISING / 1.01),
    "bc_L2p15_ramp": Workload("bc_L2p15_ramp", BLUME_CAPEL, 1 << 15, 0.0, SEED_BASE + 6, 20000,
                              1024, protocol=2, beta_f=BETA_BC / 1.01),
    # Blume-Capel at the paper's own size and temperature (Table I: L = 2^19,
    # T_c = 1.69355839821214427017, t_max = 524288): 64 GiB at 2 bits/spin -- bench.py's BC line
    "bc_L2p19": Workload("bc_L2p19", BLUME_CAPEL, 1 << 19, 0.0, SEED_BASE + 9, 524288, 4096,
                         beta_f=1.0 / 1.69355839821214427017),
    # the paper's own two-step schedules (Table II, PAPER.md:142-153;
    # the middle t_switch of each model).  Same API, a different beta array.
    "ising_L2p16_twostep": Workload("ising_L2p16_twostep", ISING, 1 << 16, 0.0, SEED_BASE + 7,
                                    3_000_000, 1024, protocol=3, beta_f=1.0 / 2.27414861561203,
                                    beta_1=1.0 / 1.66, t_switch=4467),
    "bc_L2p16_twostep": Workload("bc_L2p16_twostep", BLUME_CAPEL, 1 << 16, 0.0, SEED_BASE + 8,
                                 2_097_152, 1024, protocol=3, beta_f=1.0 / 1.69661396797728,
                                 beta_1=1.0 / 1.24, t_switch=41270),
}
