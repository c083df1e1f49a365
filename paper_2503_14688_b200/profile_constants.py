"""Numbers that come from committed ncu captures under profiles/, NOT from the current run.

bench.py's rooflines are built from the launch time it measures live; two figures can only come
from a profiler and are therefore constants taken from a capture: the thread-instructions of the
half-rate dispatch class the kernel EXECUTES per spin update, and the DRAM bytes it moves per
update.  Each entry names the profile it was read from, the commit that capture ran, and the
sha256 of the kernel sources at that commit; bench.py recomputes the hash and reports
`stale_profile: true` when the sources have changed since the capture.
"""
from __future__ import annotations

import hashlib
import os

_CSRC = os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc")

#: kernel sources whose change invalidates a capture of the model's half-sweep kernel
SOURCES = {
    0: ("philox.cuh", "ising.cuh", "ising_march.cuh"),
    1: ("philox.cuh", "ising.cuh", "ising_march.cuh", "bc.cuh", "bc_march.cuh"),
}

#: model -> constants read from the named capture
CAPTURED = {
    0: {"kernel": "ising_march_kernel",
        "executed_half_rate_instr_per_update": 3.21,      # (ALU-pipe + IMAD.WIDE/HI thread-instr) / updates, SASS page
        "dram_bytes_per_update": 0.383,                   # (dram__bytes_read + dram__bytes_write) / updates at L = 2^20
        "profile": "profiles/r2_ising_march.md + profiles/r2_launches_default.md", "commit": "628ec9c",
        "sources_sha256": "2409eae7a91bbd271cf2918bdd840392e292198010a17babc312a02761846a75"},
    1: {"kernel": "bc_march_kernel",
        "executed_half_rate_instr_per_update": 4.65,     # tables compiled in (LS >= 0); 4.77 with the dispatching kernel
        "dram_bytes_per_update": 0.768,                   # at L = 2^19 (launch list); 0.669 at L = 2^15 (partly L2-resident)
        "profile": "profiles/r2_bc_march.md + profiles/r2_launches_default.md", "commit": "628ec9c",
        "sources_sha256": "e53bde8a311852275e9e46dec8dca1350233819e23768e4f3f56738bb2de0d45"},
}

#: Algorithmic half-rate thread-instructions per update: the floor of the method under the RNG
#: contract, counted by hand in DESIGN.md section 6 (the analogue of algorithmic bytes).
ALGORITHMIC_HALF_RATE_INSTR_PER_UPDATE = {0: 2.98, 1: 4.46}
#: Algorithmic bytes per update: a half-sweep reads both colours, writes one.
ALGORITHMIC_BYTES_PER_UPDATE = {0: 0.375, 1: 0.75}


def sources_sha256(model: int) -> str:
    h = hashlib.sha256()
    for name in SOURCES[model]:
        with open(os.path.join(_CSRC, name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def captured(model: int) -> dict:
    """The model's constants plus `stale_profile` (kernel sources changed since the capture)."""
    c = dict(CAPTURED[model])
    c["stale_profile"] = c["sources_sha256"] != sources_sha256(model)
    return c
