"""The CUDA sources, executed on the CPU by a SIMT emulation, against the oracle — without a GPU.

tests/simt/ compiles paper_2606_14603_b200/csrc/ (the kernels and the C ABI's host side, as committed; three mechanical
rewrites listed in tests/simt/build.py) with g++ against a stand-in for the CUDA language and runtime in which every
CUDA thread is a fibre, warps rendezvous in __shfl / __ballot / __syncwarp, blocks in __syncthreads, mbarriers and bulk
copies follow the PTX ISA's rules, and CUDA graphs replay the recorded launches.  That is test infrastructure, not a
product path: nothing under paper_2606_14603_b200/ knows about it (checked below), and it says nothing about speed.

What it buys:
 * the bodies of the GPU parity tests (tests/test_gpu_*.py) run here, unchanged, on a machine without a GPU: the kernels'
   logic — every index, ballot, queue, barrier phase and atomic — is compared with the oracle bit for bit by the CPU tier;
 * the "device" workspace is an exactly-sized heap block filled with garbage, so an access outside it, or reliance on
   zero-initialised memory, is seen; the emulation is compiled with -DMOLSIM_CHECKS, so every data-derived index is
   also tested against its own bound (SIM_E_INTERNAL);
 * the same cases under -fsanitize=address,undefined are the memcheck that compute-sanitizer could not give on this GPU
   pool (profiles/r2_sanitizers.md), and a deliberate one-byte overrun proves that the sanitizer sees into the fibres.
The GPU tests (`-m gpu`) remain the parity tests proper: only they run the compiled SASS."""
import os
import re
import subprocess
import sys

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
sys.path[:0] = [p for p in (os.path.join(HERE, "simt"), HERE) if p not in sys.path]

import test_gpu_parity as gp  # noqa: E402
import test_gpu_readouts as gr  # noqa: E402
import test_gpu_traces as gt  # noqa: E402
import test_zz_gpu_global_tables as gz  # noqa: E402
from workloads import configs  # noqa: E402


@pytest.fixture(scope="module")
def emu():
    from harness import Emu

    return Emu(sanitize=False)


# ------------------------------------------------------------------------------------------------ it is not a product path
def test_package_does_not_know_the_emulation():
    pkg = os.path.join(ROOT, "paper_2606_14603_b200")
    for base, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(base, f), errors="replace").read()
                assert not re.search(r"simt|emulat", text, re.I), f"{f} mentions the emulation"
    for f in ("bench.py", "__graft_entry__.py"):
        assert not re.search(r"simt", open(os.path.join(ROOT, f)).read(), re.I), f


def test_rewrites_are_the_three_stated_ones():
    """The emulation build compiles the committed sources: apart from launches, dynamic shared memory declarations, one
    include path and the inline-PTX header, every line is the product's."""
    import build as simt_build

    simt_build.build()
    csrc = os.path.join(ROOT, "paper_2606_14603_b200", "csrc")
    for name in sorted(os.listdir(csrc)):
        if not name.endswith((".cu", ".cuh")) or name == "ptx_sm100.cuh":
            continue
        a = open(os.path.join(csrc, name)).read().split("\n")
        b = open(os.path.join(simt_build.OUT, "src", name.replace(".cu", ".cpp") if name.endswith(".cu") else name)).read().split("\n")
        assert len(a) == len(b), name
        for la, lb in zip(a, b):
            if la != lb:
                assert "<<<" in la or ">>>(" in la or "extern __shared__" in la or "include/molsim.h" in la, (name, la, lb)
    # the PTX header declares the same helpers on both sides
    sig = re.compile(r"inline\s+(?:__attribute__\(\(always_inline\)\)\s+)?(\w+)\s+(\w+)\(([^)]*)\)")
    prod = open(os.path.join(csrc, "ptx_sm100.cuh")).read().replace("__device__ __forceinline__", "inline")
    emu_ = open(os.path.join(HERE, "simt", "ptx_sm100_emu.cuh")).read()
    names = {m.group(2): re.sub(r"\s+", " ", m.group(3)) for m in sig.finditer(prod)}
    theirs = {m.group(2): re.sub(r"\s+", " ", m.group(3)) for m in sig.finditer(emu_)}
    assert len(names) >= 8
    for n, args in names.items():
        if n == "smem_addr":
            continue
        assert theirs.get(n) == args, (n, args, theirs.get(n))


# ------------------------------------------------------------------------------------------------ the GPU tests' bodies
@pytest.mark.parametrize("body", [
    gp.test_seeding_parity_all_geometries, gp.test_move_only_parity, gp.test_tiny_dense_cube_many_events,
    gp.test_large_displacements, gp.test_cell_size_independence_on_gpu, gp.test_channel_kinds_and_priority,
    gp.test_crowded_single_cell, gp.test_empty_population_and_mid_run_seeding, gp.test_errors,
    gt.test_homodimer_parity, gt.test_checksum_equals_oracle_and_sees_every_field,
    gt.test_w3_checkpoint_reload_with_t_first, gt.test_load_agents_rejects_bad_positions_and_duplicate_ids,
    gr.test_picture_parity_nucleus_and_cytoplasm, gr.test_compiled_compartmentalised_model_parity,
    gz.body_large_gaussian_tables, gz.body_maximum_table_sizes, gz.body_degenerate_populations,
], ids=lambda f: f.__name__)
def test_gpu_test_body_on_the_emulation(emu, body):
    body(emu)


def test_five_workload_shapes_small(emu):
    """[CFG 0-4] at sizes the emulation steps in seconds: cube, sphere cascade, replicas, (the nucleus is the checkpoint
    case above), scaling cube with a ragged population."""
    gp.run_both(emu, configs.w0(cell_size=512, n_steps=40), 40, chunks=2)
    gp.run_both(emu, configs.w1(scale=0.003, n_steps=60, cell_size=256), 60, chunks=2)
    gp.run_both(emu, configs.w2(scale=0.0005, n_steps=8, cell_size=512), 8, chunks=1)
    gp.run_both(emu, configs.w4(n=30_011, n_steps=17), 17, chunks=1)        # 17 = two 8-step graphs + one 1-step graph


@pytest.mark.parametrize("case,n_rows", [("w4_4m", 3), ("w1_full", 3), ("w3_full", 6)])
def test_full_size_oracle_traces_on_the_emulation(emu, case, n_rows):
    """BASELINE.json's sizes on the CPU tier: the first rows of the golden oracle traces (tests/golden/trace_*.txt, written by
    oracle/ only) — [CFG 4] at 4 M agents (the whole trace), [CFG 1] and [CFG 3] at full size — replayed by the emulated
    kernels: state checksum, live count, next_id, t_first and the counts row of every step.  (One-off, longer prefixes,
    [CFG 2] at full size and [CFG 4] at 64 M: profiles/r2_sanitizers.md.)"""
    import importlib.util

    spec = importlib.util.spec_from_file_location("make_traces", os.path.join(gt.GOLDEN, "make_traces.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    make = {"w4_4m": lambda: configs.w4(n=4_000_000, n_steps=2), "w1_full": lambda: configs.w1(n_steps=200),
            "w3_full": lambda: configs.w3(**mod.W3_TRACE)}[case]
    gt.replay(emu, make(), gt.read_trace(case)[:n_rows], case)


def test_graph_replay_equals_direct_launches(emu, monkeypatch):
    """sim_step replays captured graphs (the emulation records and replays the launches, parameters frozen at capture as
    on the GPU); with capture refused it issues the kernels directly.  Same result, odd and even step counts, both
    parities of the ping-pong."""
    m = gp.tiny_cube(L=301, n_a=1237, n_b=1111, p_bind=0.7, p_rel=0.05, cell=64)
    a = emu.Sim(m); a.seed_population()
    monkeypatch.setenv("SIMT_NO_GRAPHS", "1")
    b = emu.Sim(m); b.seed_population()
    for n in (1, 8, 3, 16, 5):
        a.step(n); b.step(n)
        sa, sb = a.read_agents(), b.read_agents()
        for k in sa:
            assert (sa[k] == sb[k]).all(), (n, k)
        assert (a.read_counts() == b.read_counts()).all()
    assert a.launch_count() == b.launch_count() > 0


def test_monitor_parity_small(emu):
    from oracle.monitor_view import monitor_eval

    m = gp.tiny_cube(L=301, n_a=1200, n_b=1100, p_bind=0.6, p_rel=0.01, cell=64)
    m.counts_rows = 600
    sim = emu.Sim(m); sim.seed_population(); sim.step(520)
    counts = sim.read_counts()
    Cx = 2
    plateau = int(counts[300:, 0, Cx].mean())
    mons = [dict(replica=0, species=[Cx], threshold=100, first_row=0, n_rows=521),
            dict(replica=0, species=[Cx], threshold=plateau, first_row=200, n_rows=321),
            dict(replica=0, species=[0, Cx], threshold=1199, first_row=0, n_rows=521),
            dict(replica=0, species=[0, 1, Cx, Cx], threshold=2000, first_row=520, n_rows=1)]
    gr.check_monitors(sim, counts, mons)
    assert monitor_eval(counts, 0, [0, Cx], 1199, 0, 521)["n_above"] == 521        # A + C is conserved


def test_random_models_on_the_emulation(emu, monkeypatch):
    """Parity fuzzing (tests/random_models.py): 60 seeded random models of every shape and channel mix, the second half
    under an adversarial schedule; kernels (emulated) = oracle on the full state, counts, info and checksum."""
    from paper_2606_14603_b200.binding import check_config
    from random_models import fuzz_parity

    assert fuzz_parity(emu, range(0, 30), check_config, gp.oracle_cls(), gp.assert_same) >= 26
    monkeypatch.setenv("SIMT_SCHED_SEED", "11")
    assert fuzz_parity(emu, range(30, 60), check_config, gp.oracle_cls(), gp.assert_same) >= 26


def test_random_api_sequences_on_the_emulation(emu):
    """Host-side state machine: random sequences of step(n), mid-run seeding, checkpoint reload in permuted order and
    profiling on / off, against the oracle after every call (tests/random_models.py::api_sequence_parity).  This is the
    kind of test that would have caught the build_graphs bug the emulation found."""
    from paper_2606_14603_b200.binding import check_config
    from random_models import api_sequence_parity

    assert api_sequence_parity(emu, range(0, 16), check_config, gp.oracle_cls(), gp.assert_same) >= 13


# ------------------------------------------------------------------------------------------------ sanitizers
def _asan_env():
    lib = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(lib) or not os.path.exists(lib):
        pytest.skip("libasan is not installed")
    # fake stacks (stack-use-after-return) are allocated and torn down per fibre: thousands of mmaps per launch
    env = dict(os.environ, LD_PRELOAD=lib, ASAN_OPTIONS="detect_leaks=0:detect_stack_use_after_return=0")
    env.pop("SIMT_NO_GRAPHS", None)
    return env


def test_kernels_under_address_and_ub_sanitizer():
    """The dense / crowded / large-displacement / channel / compartment / checkpoint cases with every kernel and host access
    checked by AddressSanitizer + UndefinedBehaviorSanitizer, in a child process (libasan must be preloaded)."""
    env = _asan_env()
    r = subprocess.run([sys.executable, os.path.join(HERE, "simt", "san_cases.py")], env=env, capture_output=True,
                       text=True, timeout=1500)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert "SIMT-SAN OK" in r.stdout and "ERROR: AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr


def test_kernels_under_thread_sanitizer():
    """The race check proper.  The kernels are compiled with -fsanitize=thread; every CUDA thread index is a ThreadSanitizer
    fibre, fibre switches carry no synchronisation, and happens-before exists only where CUDA gives it: launch boundaries,
    __syncthreads, __syncwarp (not shuffles or ballots), mbarrier arrive -> wait, __threadfence; atomics are relaxed
    atomics.  Shared memory is reused by the next block here, so blocks are ordered one after the other (conflicts
    between blocks are what the seeded block orders above are for).  The races the kernels have by design — K4's plain
    prop[] stores, K5's live read of t_first, same-value clears of shared bitmap words — are relaxed atomics in this build
    (tests/simt/build.py RACY_BY_DESIGN).  Anything else that two threads touch without such an edge is a report."""
    lib = subprocess.run(["gcc", "-print-file-name=libtsan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(lib) or not os.path.exists(lib):
        pytest.skip("libtsan is not installed")
    env = dict(os.environ, LD_PRELOAD=lib, TSAN_OPTIONS="halt_on_error=0 report_signal_unsafe=0 exitcode=0")
    env.pop("SIMT_NO_GRAPHS", None)
    r = subprocess.run([sys.executable, os.path.join(HERE, "simt", "san_cases.py"), "tsan"], env=env, capture_output=True,
                       text=True, timeout=1500)
    assert r.returncode == 0 and "SIMT-SAN OK" in r.stdout, r.stdout[-2000:] + r.stderr[-3000:]
    assert "ThreadSanitizer" not in r.stderr, r.stderr[:6000]


def test_sanitizer_sees_an_overrun_inside_a_kernel():
    env = _asan_env()
    r = subprocess.run([sys.executable, os.path.join(HERE, "simt", "san_cases.py"), "overrun"], env=env,
                       capture_output=True, text=True, timeout=600)
    assert r.returncode != 0 and "heap-buffer-overflow" in r.stderr and "went unnoticed" not in r.stdout


# ------------------------------------------------------------------------------------------------ schedules and races
@pytest.mark.parametrize("seed", [1])
def test_results_do_not_depend_on_the_schedule(emu, monkeypatch, seed):
    """Blocks in a random order, a random subset of the fibres in a random order on every scheduler pass, bulk copies that
    land only when somebody waits for them: the result is still the oracle's, bit for bit (every decision is keyed by id,
    min over 64-bit keys is order-free, and no kernel relies on who wins an atomic or on lock-step warps)."""
    monkeypatch.setenv("SIMT_SCHED_SEED", str(seed))
    gp.test_tiny_dense_cube_many_events(emu)
    gp.test_channel_kinds_and_priority(emu)
    gt.test_homodimer_parity(emu)
    gp.run_both(emu, configs.w4(n=30_011, n_steps=17), 17, chunks=1)
    gp.run_both(emu, configs.w3(scale=0.004, n_steps=40, cell_size=1024), 40, chunks=2)


@pytest.mark.parametrize("name,seed", [("window_keys_without_syncwarp", 0), ("tile_read_without_full_wait", 1)])
def test_a_removed_synchronisation_is_noticed(name, seed):
    """The check above has teeth (two of the five mutants of mutants.py; all five are killed, profiles/r2_sanitizers.md):
    with one synchronisation taken out of the emulation's copy of the kernels (mutants.py) the
    same cases no longer match the oracle (or trip a bound check, the deadlock report, or crash)."""
    env = dict(os.environ)
    env.pop("SIMT_NO_GRAPHS", None)
    r = subprocess.run([sys.executable, os.path.join(HERE, "simt", "mutants.py"), name, str(seed)], env=env,
                       capture_output=True, text=True, timeout=900)
    assert r.returncode != 0 and "SURVIVED" not in r.stdout, f"mutant {name} survived:\n{r.stdout[-500:]}"
