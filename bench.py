#!/usr/bin/env python
"""bench.py — molecule-agent steps/s of the whole hot path on B200 (BASELINE.json `metric`).

A "step" is one full time step (DESIGN.md §1 phases 1-6: move, boundary, spatial hash, neighbour
search + handshake, unimolecular reactions, births, compaction, counts) over the whole population.
Default workload: [CFG 4] scaling stress at N = 16 M agents (the size north_star's 60 % bar names);
`--workload w4 --n 64000000` etc. select the others.  One JSON line is printed by rank 0.

  python bench.py --gpus 1 --steps 20 --warmup 3
  python -m torch.distributed.run --nproc-per-node N ... bench.py --gpus N     (N independent replicas)
  python bench.py --impl reference          (the CPU oracle, bounded sample, rank 0 only)
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import configs  # noqa: E402

METRIC = "molecule_agent_steps_per_sec"
UNIT = "agent-steps/s"
BYTES_PER_AGENT = 18  # x,y,z int32 + id uint32 + species uint16 (north_star (1))


def make_model(args, steps_total):
    kw = {}
    if args.workload == "w4":
        kw["n"] = args.n
    elif args.scale is not None:
        kw["scale"] = args.scale
    m = configs.by_name(args.workload, **kw)
    m.counts_rows = steps_total + 2
    if args.cell_size:
        m.cell_size = args.cell_size
    elif args.workload == "w0" and args.impl != "reference":
        m.cell_size = 448      # [CFG 0]'s 5 nm cells (8 M cells for 10 k agents) are the oracle's; reading S20
    return m


def workload_name(args, m):
    if args.workload == "w4":
        return f"W4 [CFG 4] A+B<->C cube, N={args.n}, L={m.extent[0]} units, cell={m.cell_size}"
    return f"{m.name} N0={m.n_agents0} cell={m.cell_size}"


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "10", "-i", str(self.index)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._pump, daemon=True)
            self.th.start()
            t_end = time.time() + 5.0             # nvidia-smi needs a moment before its first line
            while len(self.lines) < 2 and time.time() < t_end:
                time.sleep(0.01)
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return None
        time.sleep(0.05)
        self.proc.terminate()
        # samples inside the timed region (10 ms period; a line is stamped when it is read, i.e. slightly late);
        # a region shorter than the period may hold none: then the samples nearest to it
        rows = [l.split(", ") for ts, l in self.lines if t0 <= ts <= t1 + 0.03]
        if not rows:
            near = sorted(self.lines, key=lambda e: min(abs(e[0] - t0), abs(e[0] - t1)))[:3]
            rows = [l.split(", ") for ts, l in near]
        sm, reasons, smax = [], set(), None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1])); smax = float(r[2])
            except ValueError:
                continue
            for name, v in zip(names, r[5:9]):
                if v.strip().lower() == "active":
                    reasons.add(name)
        if not sm:
            return None
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": smax, "reasons": sorted(reasons), "samples": len(sm)}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ledger_bytes_per_agent(kernel, c):
    """Algorithmic HBM bytes per live agent per launch: SURVEY.md §8(d) "Design B" column, kernel by
    kernel (DESIGN.md §5 maps each of our kernels to its row); c = cells per agent."""
    return {
        "k_uni_hist": 18 + 12 + 8 * c + 14 + 4,  # K1 (R soa, W xyz, cell count RMW) fused with K5 (resolve + unimolecular)
        "memset_cells": 0.0, "k_cell_reduce": 0.0,
        "k_cell_scan": 8 * c,                    # K2
        "k_scatter": 18 + 18 + 8 * c,            # K3: R soa, W soa, cell starts
        "k_pairs": 18 + 4 + 8 * c,               # K4: R soa, W proposal, cell starts
        "k_resolve": 0.0,
        "k_births": 0.5,                         # K6: births only + id bitmap
    }.get(kernel, 0.0)


def moved_bytes_per_agent(kernel, c):
    """What THIS implementation must move per live agent per launch: smaller than the
    §8(d) ledger where a pass was elided (move recomputed in K3, sparse proposals), larger where it keeps an
    extra array (off)."""
    return {
        "k_uni_hist": 18 + 8 * c,                # R soa once for both jobs, cell count RMW (moved positions are not stored)
        "memset_cells": 4 * c, "k_cell_reduce": 4 * c, "k_cell_scan": 8 * c,
        "k_scatter": 18 + 18 + 8 * c,            # R soa, W soa, cell cursor RMW
        "k_pairs": 18 + 0.125 + 4 * c,           # R record + species, W 1 bit; R cell starts
        "k_resolve": 0.125,                      # R proposal bitmap
    }.get(kernel, 0.0)


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """The oracle as it stands on the host cores: each step a bounded sample of the workload."""
    from oracle.binding import Oracle

    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_sample = min(args.n, args.ref_n) if args.workload == "w4" else None
    sargs = argparse.Namespace(**vars(args))
    if args.workload == "w4":
        sargs.n = n_sample
    elif args.scale is None:
        sargs.scale = 0.1
    m = make_model(sargs, args.steps + args.warmup)
    o = Oracle(m)
    o.seed_population()
    o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    c = o.read_counts()
    w, k = args.warmup, args.steps
    agent_steps = float(c[w:w + k].sum())
    val = agent_steps / dt
    full = make_model(args, 4)
    sample = (f"same recipe and density at N={m.n_agents0} agents per step (full workload N={full.n_agents0}); "
              f"{k} steps timed after {w} warm-up steps; oracle grid back end, g++ -O2")
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": k, "warmup": w, "ms_per_step": dt * 1e3 / k, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": workload_name(args, full)},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def cpu_baseline(args):
    """Oracle timed on this box's host cores on a bounded sample of the bench workload."""
    from oracle.binding import Oracle

    sargs = argparse.Namespace(**vars(args))
    if args.workload == "w4":
        sargs.n = min(args.n, args.cpu_n)
    elif args.scale is None:
        sargs.scale = 0.1
    m = make_model(sargs, 8)
    o = Oracle(m)
    o.seed_population()
    steps = max(1, args.cpu_steps)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    c = o.read_counts()
    agent_steps = float(c[:steps].sum())
    return {"value": agent_steps / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{steps} step(s) of the same recipe at N={m.n_agents0} (seeding untimed), "
                      f"{dt:.1f} s of CPU work, single thread, g++ -O2",
            "host_cpus": os.cpu_count()}


def reduce_ranks(times, work, device):
    """N independent replicas: the job's time is the MAX over ranks, its work the SUM.
    Uses whatever process group is initialised (nccl on the GPU box, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist

    tt = torch.tensor(list(times), dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    ww = torch.tensor(list(work), dtype=torch.float64, device=device)
    dist.all_reduce(ww, op=dist.ReduceOp.SUM)
    return tt.tolist(), ww.tolist()


def run_seeds(args):
    """many independent seeds of one model concurrently on one GPU, one handle and one
    CUDA stream each ("run many seeds concurrently").  Not the contract line: prints
    the aggregate agent-steps/s of R concurrent populations next to the single-population rate."""
    import torch

    import paper_2606_14603_b200 as pkg

    torch.cuda.set_device(0)
    R, W, K = args.seeds, max(3, args.warmup), args.steps
    base = make_model(args, W + 2 * K + 8)
    sims = []
    for r in range(R):
        m = make_model(args, W + 2 * K + 8)     # the first population is timed twice
        m.seed, m.place_seed = base.seed + 1000 * r, base.place_seed + 1000 * r
        s = pkg.Sim(m, device="cuda:0", stream=torch.cuda.Stream())
        s.seed_population()
        s.step(W)
        sims.append(s)
    torch.cuda.synchronize()

    def timed(group):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        main = torch.cuda.current_stream()
        ev0.record(main)
        for s in group:
            s.stream.wait_event(ev0)
        for s in group:
            s.step_async(K)
        for s in group:
            done = torch.cuda.Event()
            done.record(s.stream)
            main.wait_event(done)
        ev1.record(main)
        torch.cuda.synchronize()
        return ev0.elapsed_time(ev1)

    ms_one = timed(sims[:1])
    ms_all = timed(sims)                       # sims[0] runs K further steps: same work per step
    work = 0.0
    for s in sims:
        s.step(0)
        c = s.read_counts().astype(np.int64)
        work += float(c[-K - 1:-1].sum())
    one = float(sims[0].read_counts().astype(np.int64)[W:W + K].sum()) / (ms_one * 1e-3)
    print(json.dumps({"metric": METRIC, "unit": UNIT, "value": work / (ms_all * 1e-3), "n_gpus": 1, "steps": K,
                      "warmup": W, "ms_total": ms_all, "higher_is_better": True, "data": "synthetic", "dtype": "int32",
                      "config": {"workload": workload_name(args, base), "concurrent_seeds": R,
                                 "parallelism": f"{R} handles x 1 stream each on 1 GPU (no exchange)"},
                      "single_seed_value": one, "speedup_vs_single_seed": work / (ms_all * 1e-3) / one}), flush=True)


def run_gpu(args):
    import torch
    import torch.distributed as dist

    import paper_2606_14603_b200 as pkg

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    W, K = max(3, args.warmup), args.steps
    e2e_steps = min(K, args.e2e_steps)
    m = make_model(args, W + K + 8 + 2 * (e2e_steps + 3))
    m.seed = m.seed + rank              # replicas only: independent populations
    m.place_seed = m.place_seed + rank
    sim = pkg.Sim(m, device=f"cuda:{local}")
    sim.seed_population()
    n_cells = 1
    for a in range(3):
        n_cells *= (m.extent[a] + m.cell_size - 1) // m.cell_size

    # ---- device-resident throughput: K steps between CUDA events on the sim's stream
    sim.step(W)
    launches0 = sim.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    barrier()
    t_wall0 = time.time()
    ev0.record()
    sim.step_async(K)
    ev1.record()
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1)
    ms = ev0.elapsed_time(ev1)
    launches = sim.launch_count() - launches0
    sim.step(0)                                           # surfaces device errors
    counts = sim.read_counts(W, K + 1).astype(np.int64)
    agent_steps = float(counts[:K].sum())                 # sum_t n_live(t) over the timed steps
    n_live_mean = agent_steps / K

    # ---- per-kernel device time (events around every launch) for the roofline of the dominant kernel
    sim.profile_enable(True)
    sim.step(args.prof_steps)
    kt = sim.kernel_times()
    sim.profile_enable(False)
    step_kernels = {k: v for k, v in kt.items() if k != "other" and v[1] > 0}
    tot_ms = sum(v[0] for v in step_kernels.values())
    dom = max(step_kernels, key=lambda k: step_kernels[k][0])
    dom_ms = step_kernels[dom][0] / step_kernels[dom][1]
    c_per_agent = n_cells / n_live_mean
    peak, peak_src = measured_peak()
    n_live_prof = float(sim.read_counts(W + K, args.prof_steps).sum()) / args.prof_steps
    dom_bytes = ledger_bytes_per_agent(dom, n_cells / n_live_prof) * n_live_prof
    achieved = dom_bytes / (dom_ms * 1e-3) / 1e9
    traffic, alu = None, None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        try:
            tj = json.load(open(tpath))
            traffic = tj.get(f"{args.workload}:{args.n}", {}).get(dom)
            ipa = tj.get("warp_instr_per_agent", {}).get(f"{args.workload}:{args.n}", {}).get(dom)
            if ipa:
                # issue roofline of the dominant kernel: warp-instructions per launch (ncu count per
                # agent x live agents) / launch time, against SMs x 4 schedulers x 1 instruction per clock x SM clock
                peak_ginstr = 148 * 4 * 1.965
                ach = ipa * n_live_prof / (dom_ms * 1e-3) / 1e9
                alu = {"bound": "alu", "achieved": ach, "peak": peak_ginstr, "unit": "G warp-instr/s",
                       "frac": ach / peak_ginstr, "warp_instr_per_agent": ipa,
                       "peak_source": "148 SMs x 4 warp schedulers x 1 instr/clk x 1.965 GHz (B200_PROFILING.md clocks)"}
        except Exception:
            traffic, alu = None, None
    step_bytes = sum(ledger_bytes_per_agent(k, c_per_agent) for k in step_kernels) * n_live_mean
    moved_bytes = sum(moved_bytes_per_agent(k, c_per_agent) for k in step_kernels) * n_live_mean
    per_kernel = {k: {"ms": round(v[0] / v[1], 4), "share": round(v[0] / tot_ms, 4),
                      "ledger_gbs": round(ledger_bytes_per_agent(k, n_cells / n_live_prof) * n_live_prof /
                                          (v[0] / v[1] * 1e-3) / 1e9, 1),
                      "moved_gbs": round(moved_bytes_per_agent(k, n_cells / n_live_prof) * n_live_prof /
                                         (v[0] / v[1] * 1e-3) / 1e9, 1)}
                  for k, v in step_kernels.items()}

    # ---- end to end through the C ABI with HOST buffers: H2D of the state, one step, D2H of the counts row
    import ctypes as C
    state = sim.read_agents()
    n_host = len(state["id"])
    pinned = {k: torch.from_numpy(v.view(np.int32) if v.dtype == np.uint32 else
                                  (v.view(np.int16) if v.dtype == np.uint16 else v)).pin_memory()
              for k, v in state.items()}
    info = sim.info()
    lib = pkg.load_library()
    row = np.zeros((1, m.n_replicas, len(m.species)), dtype=np.uint32)

    def e2e_step(step_no):
        r = lib.sim_load_agents(sim._h, n_host, C.c_void_p(pinned["x"].data_ptr()), C.c_void_p(pinned["y"].data_ptr()),
                                C.c_void_p(pinned["z"].data_ptr()), C.c_void_p(pinned["species"].data_ptr()),
                                C.c_void_p(pinned["id"].data_ptr()), step_no, info["next_id"])
        assert r == 0, r
        assert lib.sim_step(sim._h, 1) == 0
        assert lib.sim_read_counts(sim._h, step_no + 1, 1, row.ctypes.data_as(C.c_void_p)) == 0
        return int(row.sum())

    base_step = info["step"]
    for i in range(2):
        e2e_step(base_step)
    barrier()
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        e2e_step(base_step)
    barrier()
    e2e_dt = time.perf_counter() - t0
    e2e_agent_steps = float(n_host) * e2e_steps

    # ---- reduce over ranks: max time, summed work
    if world > 1:
        (ms, e2e_dt), (agent_steps, e2e_agent_steps, launches) = reduce_ranks(
            [ms, e2e_dt], [agent_steps, e2e_agent_steps, float(launches)], dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    value = agent_steps / (ms * 1e-3)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32", "data": "synthetic",
        "config": {"workload": workload_name(args, m), "n_live_mean": n_live_mean,
                   "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas (no collective)",
                   "l2": "inputs larger than L2 (agent-store ping-pong %.0f MB vs 126 MB L2), no flush" %
                         (2 * BYTES_PER_AGENT * n_live_mean / 1e6),
                   "bytes_per_agent_step_ledger": round(step_bytes / n_live_mean, 1),
                   "bytes_per_agent_step_moved": round(moved_bytes / n_live_mean, 1)},
        "clocks": clocks,
        "e2e": {"value": e2e_agent_steps / e2e_dt, "unit": UNIT,
                "h2d_bytes_per_step": BYTES_PER_AGENT * n_host, "d2h_bytes_per_step": int(row.nbytes),
                "steps": e2e_steps,
                "what": "sim_load_agents(pinned host SoA) + sim_step(1) + sim_read_counts(1 row) per step"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                     "kernel_ms": dom_ms, "kernel_share_of_step": step_kernels[dom][0] / tot_ms, "alu": alu,
                     "whole_step": {"achieved": step_bytes / (ms / K * 1e-3) / 1e9,
                                    "frac": step_bytes / (ms / K * 1e-3) / 1e9 / peak,
                                    "frac_of_8TBs_nominal": step_bytes / (ms / K * 1e-3) / 1e9 / 8000.0,
                                    "moved_gbs": moved_bytes / (ms / K * 1e-3) / 1e9},
                     "per_kernel": per_kernel},
    }
    if world == 1 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(args)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="w4", choices=["w0", "w1", "w2", "w3", "w4"])
    ap.add_argument("--n", type=int, default=16_000_000, help="agents for w4")
    ap.add_argument("--scale", type=float, default=None, help="count/volume scale for w1..w3")
    ap.add_argument("--cell-size", type=int, default=0)
    ap.add_argument("--prof-steps", type=int, default=5)
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-n", type=int, default=4_000_000, help="oracle sample size for cpu_baseline")
    ap.add_argument("--cpu-steps", type=int, default=1)
    ap.add_argument("--ref-n", type=int, default=1_000_000, help="oracle sample size for --impl reference")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--seeds", type=int, default=1, help="N1: concurrent independent populations on one GPU (not the contract line)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.seeds > 1:
        run_seeds(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
