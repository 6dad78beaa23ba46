#!/usr/bin/env python
"""Writes the per-step oracle traces under tests/golden/ (checksum + counts), calling ONLY oracle/.

Full-size runs the CPU oracle cannot repeat inside the GPU test budget: the oracle is run
once here, single-threaded, and each step's order-independent 64-bit state checksum (DESIGN.md §1
"Checksum"), live count and counts row are stored; tests/test_gpu_traces.py replays the same seeded
workload on the CUDA path and compares every stored row.  No value in these files comes from the CUDA path.

  python tests/golden/make_traces.py w4_4m w4_64m w1_full w2_full w3_full      (any subset)

Line format: `t  checksum(hex)  n_live  next_id  t_first0  counts[replica][species]...` for t = 0 (after seeding) .. T.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle.binding import Oracle  # noqa: E402
from workloads import configs  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))

# case -> (model factory, steps, what it stands for)
CASES = {
    "w4_4m": (lambda: configs.w4(n=4_000_000, n_steps=2), 2, "[CFG 4] N = 4 M, scaling claim PAPER.md:107"),
    "w4_64m": (lambda: configs.w4(n=64_000_000, n_steps=1), 1, "[CFG 4] N = 64 M, scaling claim PAPER.md:107"),
    "w1_full": (lambda: configs.w1(n_steps=200), 200, "[CFG 1] full size (MAPK-shaped cascade, PAPER.md:80-97)"),
    "w2_full": (lambda: configs.w2(n_steps=20), 20, "[CFG 2] full size, 8 replicas (dose sweep, PAPER.md:80-82)"),
    "w3_full": (lambda: configs.w3(**W3_TRACE), None,
                "[CFG 3] full size, with a 50 nm gene locus, 2,000 nuclear pERK seeded at t = 0 and the repressor delay "
                "shortened to 200 steps so that gene binding, transcription and the delayed rule all happen "
                "inside the trace (cFos expression, PAPER.md:153-167; workloads/configs.py w3)"),
}
W3_TRACE = dict(n_steps=800, delay=200, gene_radius=500, primed_perk_n=2000)


def run(case):
    make, steps, what = CASES[case]
    m = make()
    steps = m.n_steps if steps is None else steps
    m.counts_rows = steps + 2
    o = Oracle(m)
    o.seed_population()
    path = os.path.join(HERE, f"trace_{case}.txt")
    t0 = time.time()
    with open(path + ".tmp", "w") as f:
        f.write(f"# oracle trace {case}: {what}\n")
        f.write(f"# model {m.name}, N0 = {m.n_agents0}, seed {m.seed}, place_seed {m.place_seed}, cell_size {m.cell_size} "
                f"(results do not depend on it, S20), {steps} steps\n")
        f.write("# written by tests/golden/make_traces.py from oracle/ only (single thread); columns: t checksum n_live "
                "next_id t_first0 counts...\n")
        for t in range(steps + 1):
            if t:
                o.step(1)
            info = o.info()
            row = o.read_counts(t, 1).reshape(-1)
            f.write(f"{t} {o.read_checksum():016x} {info['n_live']} {info['next_id']} {info['t_first0']} "
                    + " ".join(str(int(v)) for v in row) + "\n")
            f.flush()
            if t % 50 == 0:
                print(f"{case}: t={t} n_live={info['n_live']} t_first0={info['t_first0']} {time.time() - t0:.0f}s", flush=True)
    os.replace(path + ".tmp", path)
    print(f"{case}: wrote {path} in {time.time() - t0:.0f}s")


if __name__ == "__main__":
    for c in sys.argv[1:] or list(CASES):
        run(c)
