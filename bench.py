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


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def kernel_source_hash():
    """sha256 over the CUDA sources: profiles/traffic.json is stamped with it, so ncu-derived constants (DRAM traffic,
    warp instructions per agent) are only quoted for the kernels they were measured on."""
    import hashlib

    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2606_14603_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh")):
            h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


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
def oracle_sample_model(args, steps_total):
    """The ONE bounded sample both oracle legs time: the bench workload's recipe at a size the single-threaded oracle
    gets through in tens of seconds ([CFG 4]: same density, N <= --oracle-n; the sphere workloads: --scale 0.1)."""
    sargs = argparse.Namespace(**vars(args))
    if args.workload == "w4":
        sargs.n = min(args.n, args.oracle_n)
    elif args.scale is None:
        sargs.scale = 0.1
    return make_model(sargs, steps_total)


def time_oracle(args, warmup, steps):
    from oracle.binding import Oracle

    m = oracle_sample_model(args, warmup + steps + 2)
    o = Oracle(m)
    o.seed_population()
    o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    c = o.read_counts()
    agent_steps = float(c[warmup:warmup + steps].sum())
    full = make_model(args, 4)
    sample = (f"{steps} step(s) after {warmup} untimed, same recipe and density at N0={m.n_agents0} "
              f"(bench workload N0={full.n_agents0}); {dt:.1f} s of CPU work; oracle grid back end, 1 thread, g++ -O2")
    return {"value": agent_steps / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
            "host_cpus": os.cpu_count(), "cpu_model": cpu_model()}, dt, m


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, on the bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cb, dt, m = time_oracle(args, args.warmup, args.steps)
    line = {
        "impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": workload_name(argparse.Namespace(**{**vars(args), "n": m.n_agents0}), m) +
                               f" (bounded sample of the bench workload; what ran: N0={m.n_agents0})"},
        "cpu_baseline": cb,
        "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def cpu_baseline(args):
    """Oracle timed on this box's host cores on the same bounded sample --impl reference uses."""
    return time_oracle(args, 1, max(1, args.cpu_steps))[0]


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


def n_cells_of(m):
    n = 1
    for a in range(3):
        n *= (m.extent[a] + m.cell_size - 1) // m.cell_size
    return n


def step_fractions(step_kernels_names, n_cells, n_live_mean, ms_per_step, peak):
    c = n_cells / n_live_mean
    ledger = sum(ledger_bytes_per_agent(k, c) for k in step_kernels_names) * n_live_mean
    moved = sum(moved_bytes_per_agent(k, c) for k in step_kernels_names) * n_live_mean
    gbs = ledger / (ms_per_step * 1e-3) / 1e9
    return {"bytes_per_agent_step_ledger": round(ledger / n_live_mean, 1),
            "bytes_per_agent_step_moved": round(moved / n_live_mean, 1),
            "ledger_gbs": gbs, "frac_of_measured_peak": gbs / peak, "frac_of_8TBs_nominal": gbs / 8000.0,
            "moved_gbs": moved / (ms_per_step * 1e-3) / 1e9, "moved_frac_of_measured_peak": moved / (ms_per_step * 1e-3) / 1e9 / peak}


STEP_KERNELS = ["memset_cells", "k_cell_reduce", "k_cell_scan", "k_scatter", "k_pairs", "k_resolve", "k_uni_hist", "k_births"]


def run_sweep(args, pkg, torch, local, peak):
    """Short device-timed runs of the rest of the metric's range (BASELINE.json: "at 1M-64M agents", five workloads) so
    that the driver's record, not prose, holds them: a few steps each, CUDA events, clocks sampled per run."""
    out = []
    cases = [("w0", {}), ("w1", {}), ("w2", {}), ("w3", {}), ("w4", {"n": 1_000_000}), ("w4", {"n": 4_000_000}),
             ("w4", {"n": 64_000_000})]
    for wl, kw in cases:
        if wl == args.workload and kw.get("n", args.n) == args.n:
            continue
        a2 = argparse.Namespace(**{**vars(args), "workload": wl, "n": kw.get("n", args.n), "scale": None, "cell_size": 0})
        W, K = 5, (200 if wl in ("w0", "w3") else 20)
        m = make_model(a2, W + K + 4)
        sim = pkg.Sim(m, device=f"cuda:{local}")
        sim.seed_population()
        sim.step(W)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(local)
        sampler.start()
        torch.cuda.synchronize()
        t0 = time.time()
        ev0.record()
        sim.step_async(K)
        ev1.record()
        torch.cuda.synchronize()
        t1 = time.time()
        clocks = sampler.stop(t0, t1)
        ms = ev0.elapsed_time(ev1)
        sim.step(0)
        agent_steps = float(sim.read_counts(W, K).astype(np.int64).sum())
        fr = step_fractions(STEP_KERNELS, n_cells_of(m), agent_steps / K, ms / K, peak)
        out.append({"workload": workload_name(a2, m), "steps": K, "ms_per_step": ms / K,
                    "value": agent_steps / (ms * 1e-3), "n_live_mean": agent_steps / K,
                    "ledger_frac_of_measured_peak": round(fr["frac_of_measured_peak"], 4),
                    "ledger_frac_of_8TBs_nominal": round(fr["frac_of_8TBs_nominal"], 4),
                    "moved_gbs": round(fr["moved_gbs"], 1), "clocks": clocks})
        sim.close()
        del sim
        torch.cuda.empty_cache()
    return out


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

    W, K, R, SETTLE = max(3, args.warmup), args.steps, max(1, args.repeats), 3
    e2e_steps = min(K, args.e2e_steps)
    m = make_model(args, W + SETTLE + K + args.prof_steps + 8)
    m.seed = m.seed + rank              # replicas only: independent populations
    m.place_seed = m.place_seed + rank
    sim = pkg.Sim(m, device=f"cuda:{local}")
    sim.seed_population()
    n_cells = n_cells_of(m)
    peak, peak_src = measured_peak()

    # ---- the state every repeat starts from: W warm-up steps, then read back into pinned host memory
    import ctypes as C
    sim.step(W)
    state = sim.read_agents()
    n_host = len(state["id"])
    pinned = {k: torch.from_numpy(v.view(np.int32) if v.dtype == np.uint32 else
                                  (v.view(np.int16) if v.dtype == np.uint16 else v)).pin_memory()
              for k, v in state.items()}
    info = sim.info()
    lib = pkg.load_library()

    def reload_state():
        r = lib.sim_load_agents(sim._h, n_host, C.c_void_p(pinned["x"].data_ptr()), C.c_void_p(pinned["y"].data_ptr()),
                                C.c_void_p(pinned["z"].data_ptr()), C.c_void_p(pinned["species"].data_ptr()),
                                C.c_void_p(pinned["id"].data_ptr()), info["step"], info["next_id"])
        assert r == 0, r

    # ---- device-resident throughput: R repeats, each from the same reloaded state: SETTLE untimed steps (the reload
    # hands the agents over in id order; the first sort puts them back in cell order), then K steps between CUDA events
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    t_wall0 = time.time()
    rep_ms, rep_work, launches = [], [], 0
    for r in range(R):
        reload_state()
        sim.step(SETTLE)
        launches0 = sim.launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record()
        sim.step_async(K)
        ev1.record()
        barrier()
        rep_ms.append(ev0.elapsed_time(ev1))
        launches = sim.launch_count() - launches0
        sim.step(0)                                           # surfaces device errors
        counts = sim.read_counts(W + SETTLE, K + 1).astype(np.int64)
        rep_work.append(float(counts[:K].sum()))              # sum_t n_live(t) over the timed steps
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1)

    # ---- per-kernel device time (events around every launch) for the roofline of the dominant kernel
    sim.profile_enable(True)
    sim.step(args.prof_steps)
    kt = sim.kernel_times()
    sim.profile_enable(False)
    step_kernels = {k: v for k, v in kt.items() if k not in ("other", "k_hist_prologue") and v[1] > 0}
    tot_ms = sum(v[0] for v in step_kernels.values())
    dom = max(step_kernels, key=lambda k: step_kernels[k][0])
    dom_ms = step_kernels[dom][0] / step_kernels[dom][1]
    n_live_prof = float(sim.read_counts(W + SETTLE + K, args.prof_steps).sum()) / args.prof_steps
    c_prof = n_cells / n_live_prof
    per_kernel = {k: {"ms": round(v[0] / v[1], 4), "share": round(v[0] / tot_ms, 4),
                      "ledger_gbs": round(ledger_bytes_per_agent(k, c_prof) * n_live_prof / (v[0] / v[1] * 1e-3) / 1e9, 1),
                      "moved_gbs": round(moved_bytes_per_agent(k, c_prof) * n_live_prof / (v[0] / v[1] * 1e-3) / 1e9, 1)}
                  for k, v in step_kernels.items()}

    # ncu-derived constants of the dominant kernel (DRAM bytes and warp instructions per launch), quoted only while the
    # CUDA sources are the ones they were measured on (profiles/traffic.json carries their hash)
    traffic, ipa, traffic_src = None, None, None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    src_hash = kernel_source_hash()
    if os.path.exists(tpath):
        try:
            tj = json.load(open(tpath))
            if tj.get("source_sha16") == src_hash:
                ent = tj.get(f"{args.workload}:{args.n}", {}).get(dom)
                if ent:
                    traffic, ipa, traffic_src = ent.get("dram_bytes"), ent.get("warp_instr_per_agent"), tj.get("profile")
        except Exception:
            pass

    # ---- end to end through the C ABI with HOST buffers: H2D of the state, one step, D2H of the counts row
    row = np.zeros((1, m.n_replicas, len(m.species)), dtype=np.uint32)

    def e2e_step():
        reload_state()
        assert lib.sim_step(sim._h, 1) == 0
        assert lib.sim_read_counts(sim._h, info["step"] + 1, 1, row.ctypes.data_as(C.c_void_p)) == 0
        return int(row.sum())

    for i in range(2):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        e2e_step()
    barrier()
    e2e_dt = time.perf_counter() - t0
    e2e_agent_steps = float(n_host) * e2e_steps

    # ---- reduce over ranks: max time per repeat, summed work
    if world > 1:
        tt, ww = reduce_ranks(rep_ms + [e2e_dt], rep_work + [e2e_agent_steps, float(launches)], dev)
        rep_ms, e2e_dt = tt[:R], tt[R]
        rep_work, e2e_agent_steps, launches = ww[:R], ww[R], ww[R + 1]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    rates = [w / (t * 1e-3) for w, t in zip(rep_work, rep_ms)]
    med = int(np.argsort(rates)[len(rates) // 2])          # the median repeat
    ms, agent_steps, value = rep_ms[med], rep_work[med], rates[med]
    n_live_mean = agent_steps / K / world
    fr = step_fractions(list(step_kernels), n_cells, n_live_mean, ms / K, peak)

    # roofline of the dominant kernel.  k_pairs is bound by integer instruction issue, not by HBM:
    # with ncu's instruction count of the same sources it is reported against the issue peak, else by its ledger bytes
    if ipa:
        peak_ginstr = 148 * 4 * 1.965
        ach = ipa * n_live_prof / (dom_ms * 1e-3) / 1e9
        roof = {"bound": "alu", "kernel": dom, "achieved": ach, "peak": peak_ginstr, "unit": "G warp-instr/s",
                "frac": ach / peak_ginstr, "traffic": traffic,
                "peak_source": "148 SMs x 4 warp schedulers x 1 instr/clk x 1.965 GHz (B200_PROFILING.md clocks; DESIGN.md §6)",
                "warp_instr_per_agent": ipa, "ncu_profile": traffic_src}
    else:
        dom_bytes = ledger_bytes_per_agent(dom, c_prof) * n_live_prof
        ach = dom_bytes / (dom_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": None, "peak_source": peak_src,
                "note": "no ncu constants for these sources (profiles/traffic.json hash differs): ledger bytes / event time"}
    roof.update({"kernel_ms": dom_ms, "kernel_share_of_step": step_kernels[dom][0] / tot_ms,
                 "hbm_ledger_gbs": round(ledger_bytes_per_agent(dom, c_prof) * n_live_prof / (dom_ms * 1e-3) / 1e9, 1),
                 "whole_step": {"achieved": fr["ledger_gbs"], "frac": fr["frac_of_measured_peak"],
                                "frac_of_8TBs_nominal": fr["frac_of_8TBs_nominal"], "moved_gbs": fr["moved_gbs"],
                                "moved_frac": fr["moved_frac_of_measured_peak"], "peak": peak, "peak_source": peak_src,
                                "what": "ledger = SURVEY 8(d) Design B bytes / device time (the contract's number); moved = the "
                                        "bytes this implementation has to move (DESIGN.md §6): the honest companion"},
                 "per_kernel": per_kernel,
                 "per_kernel_note": "k_uni_hist's ledger charges K1 + K5 of the survey (48 B + 8c per agent); it moves 18 B + 8c"})
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32", "data": "synthetic",
        "config": {"workload": workload_name(args, m), "n_live_mean": n_live_mean,
                   "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas (no collective)",
                   "l2": "inputs larger than L2 (agent-store ping-pong %.0f MB vs 126 MB L2), no flush" %
                         (2 * BYTES_PER_AGENT * n_live_mean / 1e6),
                   "bytes_per_agent_step_ledger": fr["bytes_per_agent_step_ledger"],
                   "bytes_per_agent_step_moved": fr["bytes_per_agent_step_moved"],
                   "kernel_source_sha16": src_hash},
        "repeats": {"n": R, "what": f"each repeat: sim_load_agents of the same state (step {info['step']}), {SETTLE} untimed steps, "
                                    f"{K} timed steps; value = median repeat",
                    "ms_per_step": [round(t / K, 5) for t in rep_ms], "spread": (max(rates) - min(rates)) / value},
        "clocks": clocks,
        "e2e": {"value": e2e_agent_steps / e2e_dt, "unit": UNIT,
                "h2d_bytes_per_step": BYTES_PER_AGENT * n_host, "d2h_bytes_per_step": int(row.nbytes),
                "steps": e2e_steps,
                "what": "sim_load_agents(pinned host SoA) + sim_step(1) + sim_read_counts(1 row) per step"},
        "gpu_launches": int(launches),
        "roofline": roof,
    }
    if world == 1 and not args.no_sweep:
        sim.close()
        del sim
        torch.cuda.empty_cache()
        line["sweep"] = run_sweep(args, pkg, torch, local, peak)
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
    ap.add_argument("--oracle-n", type=int, default=1_000_000, help="agents of the bounded sample both oracle legs time (w4)")
    ap.add_argument("--cpu-steps", type=int, default=5, help="timed oracle steps of the cpu_baseline leg")
    ap.add_argument("--repeats", type=int, default=5, help="timed repeats from the same reloaded state (median reported)")
    ap.add_argument("--no-sweep", action="store_true", help="skip the short runs of the other workloads / sizes")
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
