"""The N > 1 path of bench.py on CPU (gloo, world size 2): replicas only, so the only cross-rank logic is
max-over-ranks time / summed work and "rank 0 alone runs the reference arm"."""
import json
import os
import socket
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    times, work = bench.reduce_ranks([1.0 + rank, 5.0 - rank], [100.0 * (rank + 1), 7.0, 220.0], torch.device("cpu"))
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, times, work))


def test_reduce_ranks_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, times, work in out:
        assert times == [2.0, 5.0]            # max over ranks, per entry
        assert work == [300.0, 14.0, 440.0]   # summed over ranks


def test_reference_arm_rank1_exits_without_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_rank0_prints_contract_line():
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "1", "--oracle-n", "20000"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "molecule_agent_steps_per_sec"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert "N=20000" in line["config"]["workload"] and line["cpu_baseline"]["cpu_model"]   # names what actually ran


def test_ncu_constants_are_quoted_only_for_the_sources_they_were_measured_on():
    """profiles/traffic.json carries a sha256 of paper_2606_14603_b200/csrc; bench.py recomputes it and drops the
    ncu-derived fields (roofline.traffic, warp instructions per agent) when the sources have changed since."""
    sys.path.insert(0, ROOT)
    import bench

    tj = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    assert len(tj["source_sha16"]) == 16 and tj["profile"].startswith("profiles/")
    ent = tj["w4:16000000"]["k_pairs"]
    assert ent["dram_bytes"] > 0 and 5.0 < ent["warp_instr_per_agent"] < 15.0
    # the committed capture belongs to the committed kernels (a kernel change must come with a new capture, or the
    # bench line falls back to ledger bytes and says so)
    assert bench.kernel_source_hash() == tj["source_sha16"]


def test_ledger_and_moved_bytes_per_agent_step():
    """SURVEY.md 8(d) Design B: 106.5 + 32c bytes per agent-step over the step's kernels; what the implementation moves
    is smaller."""
    sys.path.insert(0, ROOT)
    import bench

    c = 0.25
    ledger = sum(bench.ledger_bytes_per_agent(k, c) for k in bench.STEP_KERNELS)
    assert abs(ledger - (106.5 + 32 * c)) < 1e-9
    moved = sum(bench.moved_bytes_per_agent(k, c) for k in bench.STEP_KERNELS)
    assert abs(moved - (18 + 8 * c + 4 * c + 4 * c + 8 * c + 36 + 8 * c + 18.125 + 4 * c + 0.125)) < 1e-9 and moved < ledger
    fr = bench.step_fractions(bench.STEP_KERNELS, 1_000_000, 4_000_000.0, 1.0, 6532.2)
    assert abs(fr["ledger_gbs"] - (106.5 + 8) * 4e6 / 1e-3 / 1e9) < 1e-6
    assert abs(fr["frac_of_8TBs_nominal"] - fr["ledger_gbs"] / 8000.0) < 1e-12
