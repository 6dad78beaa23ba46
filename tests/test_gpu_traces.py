"""GPU parity at the sizes and lengths the CPU oracle cannot repeat inside a test: the CUDA path is replayed step by
step against the oracle traces under tests/golden/ (tests/golden/make_traces.py wrote them from oracle/ only).

Every stored row is compared: the order-independent 64-bit checksum of the live (id, species, x, y, z)
(DESIGN.md §1 "Checksum": it stands in for the element-by-element comparison), the live count, next_id, the first
delayed rule's t_first and the whole counts row.  Integer work, so the bar is equality.  Covers north_star's
"bit-exact agreement with the CPU oracle on all five configs" for [CFG 4] at 4 M and 64 M, [CFG 1]
and [CFG 2] at full size over 200 / 20 steps and [CFG 3] at full size through first transcription + the delayed
repressor.  Also here: checksum / checkpoint / homodimer parity against the live oracle.
"""
import os

import numpy as np
import pytest

from workloads import configs
from workloads.model import (CH_RELEASE, SHAPE_CUBE, Channel, Compartment, Model, Reaction, SeedRecord, Species,
                             prob_to_thr, stack_tables)

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module")
def gpu():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_14603_b200 as pkg

    pkg.load_library()
    return pkg


def read_trace(case):
    path = os.path.join(GOLDEN, f"trace_{case}.txt")
    rows = []
    with open(path) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            p = line.split()
            rows.append((int(p[0]), int(p[1], 16), int(p[2]), int(p[3]), int(p[4]), np.array(p[5:], dtype=np.int64)))
    return rows


def replay(gpu, m, rows, what):
    m.counts_rows = len(rows) + 1
    sim = gpu.Sim(m)
    sim.seed_population()
    for t, chk, n_live, next_id, t_first0, counts in rows:
        if t:
            sim.step(1)
        info = sim.info()
        assert info["step"] == t
        assert (info["n_live"], info["next_id"], info["t_first0"]) == (n_live, next_id, t_first0), (what, t, info)
        assert sim.read_checksum() == chk, f"{what}: state checksum differs from the oracle's at step {t}"
    got = sim.read_counts().astype(np.int64).reshape(len(rows), -1)
    want = np.stack([r[5] for r in rows])
    bad = np.nonzero((got != want).any(axis=1))[0]
    assert len(bad) == 0, f"{what}: counts differ first at row {bad[0]}"
    return sim


@pytest.mark.parametrize("case,make", [
    ("w4_4m", lambda: configs.w4(n=4_000_000, n_steps=2)),
    ("w4_64m", lambda: configs.w4(n=64_000_000, n_steps=1)),
    ("w1_full", lambda: configs.w1(n_steps=200)),
    ("w2_full", lambda: configs.w2(n_steps=20)),
])
def test_full_size_runs_follow_the_oracle_trace(gpu, case, make):
    rows = read_trace(case)
    replay(gpu, make(), rows, case)


def test_w3_full_size_expression_follows_the_oracle_trace(gpu):
    """[CFG 3] at full size through gene binding, first transcription and the delayed repressor."""
    import importlib.util

    spec = importlib.util.spec_from_file_location("make_traces", os.path.join(GOLDEN, "make_traces.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    W3_TRACE = mod.W3_TRACE

    rows = read_trace("w3_full")
    m = configs.w3(**W3_TRACE)
    sim = replay(gpu, m, rows, "w3_full")
    ix = {s.name: i for i, s in enumerate(m.species)}
    c = np.stack([r[5] for r in rows])
    t_first = rows[-1][4]
    assert t_first != 0xFFFFFFFF and t_first + W3_TRACE["delay"] < len(rows) - 1      # the trace covers the delayed rule
    assert c[:, ix["mRNA_n"]].max() > 0 and c[:, ix["GENE:pERK"]].max() > 0           # gene bound, transcription
    born = t_first + W3_TRACE["delay"] + 1                                            # row after the step that emits F_n
    assert c[born - 1, ix["F_n"]] + c[born - 1, ix["GENE:F"]] == 0
    assert c[born, ix["F_n"]] + c[born, ix["GENE:F"]] == 2                            # one repressor per gene locus
    assert (c[:, ix["GENE"]] + c[:, ix["GENE:pERK"]] + c[:, ix["GENE:F"]] == 2).all()
    assert sim.info()["t_first0"] == t_first


# ------------------------------------------------------------------------------------------------ live oracle
def oracle_cls():
    from oracle.binding import Oracle

    return Oracle


def same_state(sim, orc, what):
    a, b = sim.read_agents(), orc.read_agents()
    for k in ("id", "species", "x", "y", "z"):
        assert len(a[k]) == len(b[k]) and (a[k] == b[k]).all(), (what, k)
    assert (sim.read_counts() == orc.read_counts()).all(), what
    assert sim.read_checksum() == orc.read_checksum(), what
    assert sim.info() == orc.info(), what
    assert (sim.read_t_first() == orc.read_t_first()).all(), what


def test_checksum_equals_oracle_and_sees_every_field(gpu):
    m = configs.w4(n=200_000, n_steps=8)
    sim, orc = gpu.Sim(m), oracle_cls()(m)
    sim.seed_population(); orc.seed_population()
    seen = set()
    for t in range(6):
        assert sim.read_checksum() == orc.read_checksum(), t
        seen.add(sim.read_checksum())
        sim.step(1); orc.step(1)
    assert len(seen) == 6
    a = sim.read_agents()
    base = sim.read_checksum()
    info = sim.info()
    for k in ("x", "y", "z", "species", "id"):                 # a one-unit change of any field of one agent shows
        b = {f: v.copy() for f, v in a.items()}
        if k == "id":
            b[k][-1] = info["next_id"]
        elif k == "species":
            b[k][7] = (b[k][7] + 1) % 3
        else:
            b[k][7] = b[k][7] + 1 if b[k][7] + 1 < m.extent[0] else b[k][7] - 1
        sim.load_agents(b["x"], b["y"], b["z"], b["species"], b["id"], step=info["step"], next_id=info["next_id"] + 1)
        assert sim.read_checksum() != base, k
    perm = np.random.default_rng(1).permutation(len(a["id"]))  # ... and the order of the agents does not
    sim.load_agents(*(a[k][perm] for k in ("x", "y", "z", "species", "id")), step=info["step"], next_id=info["next_id"])
    assert sim.read_checksum() == base


def test_homodimer_parity(gpu):
    """A + A -> D with the smaller id as anchor (reading S10), D -> A + A release; dense, so many mutual pairs."""
    A, D = 0, 1
    m = Model(name="homodimer", species=[Species("A", 1), Species("D", 2, channels=[Channel(CH_RELEASE, prob_to_thr(0.05), A, A)])],
              reactions=[Reaction(A, A, D, 2500, prob_to_thr(0.6))], compartments=[Compartment(SHAPE_CUBE, L=500)],
              table_bits=12, tables=stack_tables([44.7214, 31.6228], 12), extent=(500,) * 3, seed=77, place_seed=78,
              seed_records=[SeedRecord(A, 6000)], n_steps=40, cell_size=100).finalize()
    sim, orc = gpu.Sim(m), oracle_cls()(m)
    sim.seed_population(); orc.seed_population()
    for chunk in range(4):
        sim.step(10); orc.step(10)
        same_state(sim, orc, f"homodimer after {(chunk + 1) * 10} steps")
    c = orc.read_counts()[:, 0, :].astype(np.int64)
    assert c[:, D].max() > 500 and (c[:, A] + 2 * c[:, D] == 6000).all()


def test_w3_checkpoint_reload_with_t_first(gpu):
    """state = (agents, t, next_id, t_first[]): save at step a into a FRESH handle, step b, and get
    step(a + b) bit for bit, delayed repressor included."""
    kw = dict(scale=0.02, n_steps=400, delay=60, gene_radius=500, primed_perk_n=400)
    m = configs.w3(**kw)
    ref = gpu.Sim(m); ref.seed_population()
    orc = oracle_cls()(m); orc.seed_population()
    t_save = None
    for t in range(0, 300, 10):
        ref.step(10); orc.step(10)
        if ref.info()["t_first0"] != 0xFFFFFFFF:
            t_save = ref.info()["step"]
            break
    assert t_save is not None, "no transcription in 300 steps: pick other parameters"
    same_state(ref, orc, "w3 before the checkpoint")
    a, info, tf = ref.read_agents(), ref.info(), ref.read_t_first()
    assert tf[0] + kw["delay"] >= t_save                       # the delayed rule has NOT fired yet: it must survive the reload
    left = int(tf[0]) + kw["delay"] + 20 - t_save
    fresh = gpu.Sim(configs.w3(**kw))
    fresh.load_agents(a["x"], a["y"], a["z"], a["species"], a["id"], step=info["step"], next_id=info["next_id"])
    fresh.load_t_first(tf)
    o2 = oracle_cls()(configs.w3(**kw))
    o2.load_agents(a["x"], a["y"], a["z"], a["species"], a["id"], step=info["step"], next_id=info["next_id"])
    o2.load_t_first(tf)
    ref.step(left); orc.step(left); fresh.step(left); o2.step(left)
    same_state(ref, orc, "w3 uninterrupted")
    fa, ra = fresh.read_agents(), ref.read_agents()
    for k in fa:
        assert (fa[k] == ra[k]).all(), k
    assert fresh.read_checksum() == ref.read_checksum() == o2.read_checksum()
    ix = {s.name: i for i, s in enumerate(m.species)}
    c = fresh.read_counts(info["step"], left + 1)[:, 0, :].astype(np.int64)
    assert (c[:, ix["F_n"]] + c[:, ix["GENE:F"]]).max() == 2   # the repressor was born in the reloaded handle
    assert (c == ref.read_counts(info["step"], left + 1)[:, 0, :]).all()


def test_load_agents_rejects_bad_positions_and_duplicate_ids(gpu):
    from paper_2606_14603_b200.binding import E_INVAL

    m = configs.w3(scale=0.02, n_steps=8)
    sim = gpu.Sim(m); sim.seed_population()
    a, info = sim.read_agents(), sim.info()
    n = len(a["id"])

    def load(**over):
        b = {k: v.copy() for k, v in a.items()}
        for k, (i, v) in over.items():
            b[k][i] = v
        return sim._lib.sim_load_agents(sim._h, n, *(b[k].ctypes.data for k in ("x", "y", "z", "species", "id")),
                                        info["step"], info["next_id"])

    assert load() == 0
    assert load(y=(5, -3)) == E_INVAL                       # negative coordinate
    assert load(z=(5, m.extent[2] + 1000)) == E_INVAL       # beyond the extent
    assert load(id=(5, int(a["id"][6]))) == E_INVAL         # duplicate id
    assert load(id=(5, info["next_id"])) == E_INVAL         # id not below next_id
    assert load(species=(5, len(m.species))) == E_INVAL     # unknown species
    # a cytoplasmic agent placed at the centre of the nucleus: valid coordinates, wrong compartment
    cyt = int(np.nonzero(np.array([s.compartment for s in m.species])[a["species"]] == 0)[0][0])
    c0 = m.compartments[0]
    b = {k: v.copy() for k, v in a.items()}
    b["x"][cyt], b["y"][cyt], b["z"][cyt] = c0.cx, c0.cy, c0.cz
    assert sim._lib.sim_load_agents(sim._h, n, *(b[k].ctypes.data for k in ("x", "y", "z", "species", "id")),
                                    info["step"], info["next_id"]) == E_INVAL
    assert sim.info()["n_live"] == 0                            # an EMPTY, usable population is left behind
    assert load() == 0 and sim.info()["n_live"] == n
    sim.step(2)                                                 # ... and the handle still steps
