"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit-exact.

Every comparison is element by element on id-sorted agent states and on the full per-step
counts log, on the same seeded synthetic inputs (north_star: "bit-exactly on the same seeded
inputs").  Integer work only, so the bar is equality.
"""
import numpy as np
import pytest

from workloads import configs
from workloads.model import (CH_BIRTH, CH_CONVERT, CH_DEGRADE, CH_RELEASE, SHAPE_CUBE, Channel,
                             Compartment, Model, Reaction, SeedRecord, Species, prob_to_thr,
                             stack_tables)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_14603_b200 as pkg

    pkg.load_library()          # fails loudly if the extension is missing
    return pkg


def oracle_cls():
    from oracle.binding import Oracle

    return Oracle


def assert_same(sim, orc, what=""):
    a, b = sim.read_agents(), orc.read_agents()
    assert len(a["id"]) == len(b["id"]), f"{what}: live count {len(a['id'])} vs oracle {len(b['id'])}"
    for k in ("id", "species", "x", "y", "z"):
        bad = np.nonzero(a[k] != b[k])[0]
        assert len(bad) == 0, f"{what}: {k} differs at {len(bad)} agents, first id {b['id'][bad[0]]}"
    ca, cb = sim.read_counts(), orc.read_counts()
    assert ca.shape == cb.shape
    bad = np.nonzero((ca != cb).any(axis=(1, 2)))[0]
    assert len(bad) == 0, f"{what}: counts differ first at row {bad[0]}"
    ia, ib = sim.info(), orc.info()
    assert ia == ib, f"{what}: info {ia} vs {ib}"


def run_both(gpu, m, steps, chunks=1, cell_gpu=None, cell_orc=None):
    sim = gpu.Sim(m, cell_size=cell_gpu)
    orc = oracle_cls()(m, cell_size=cell_orc)
    sim.seed_population(); orc.seed_population()
    assert_same(sim, orc, f"{m.name} seeding")
    per = steps // chunks
    for c in range(chunks):
        sim.step(per); orc.step(per)
        assert_same(sim, orc, f"{m.name} after {(c + 1) * per} steps")
    return sim, orc


def tiny_cube(L=400, n_a=1000, n_b=1000, p_bind=0.5, p_rel=1e-3, cell=64, seed=11):
    A, B, Cx = 0, 1, 2
    m = Model(
        name="tiny", species=[Species("A", 1), Species("B", 1),
                              Species("C", 2, channels=[Channel(CH_RELEASE, prob_to_thr(p_rel), A, B)])],
        reactions=[Reaction(A, B, Cx, 2500, prob_to_thr(p_bind))],
        compartments=[Compartment(SHAPE_CUBE, L=L)], table_bits=12, tables=stack_tables([44.7214, 31.6228], 12),
        extent=(L, L, L), seed=seed, place_seed=seed,
        seed_records=[SeedRecord(A, n_a), SeedRecord(B, n_b)], n_steps=64, cell_size=cell)
    return m.finalize()


# ------------------------------------------------------------------------------------------------
def test_philox_device_equals_oracle_and_torch(gpu, torch_philox):
    from oracle.binding import philox
    from paper_2606_14603_b200.binding import debug_philox

    rng = np.random.default_rng(7)
    n = 200_000
    ctr = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0; key[0] = 0; ctr[1] = 0xFFFFFFFF; key[1] = 0xFFFFFFFF
    dev = debug_philox(ctr, key)
    assert (dev == torch_philox(ctr, key)).all()                  # library routine
    for i in range(0, 2000):
        assert (dev[i] == philox(ctr[i], key[i])).all()           # oracle


def test_seeding_parity_all_geometries(gpu):
    for m in (configs.w0(), configs.w1(scale=0.02), configs.w2(scale=0.004), configs.w3(scale=0.05)):
        sim = gpu.Sim(m); orc = oracle_cls()(m)
        sim.seed_population(); orc.seed_population()
        assert_same(sim, orc, m.name)


def test_move_only_parity(gpu):
    for m in (tiny_cube(L=300), configs.w3(scale=0.02), configs.w2(scale=0.002)):
        sim = gpu.Sim(m); orc = oracle_cls()(m)
        sim.seed_population(); orc.seed_population()
        sim.debug_move_only(); orc.debug_move_only()
        a, b = sim.read_agents(), orc.read_agents()
        for k in ("id", "species", "x", "y", "z"):
            assert (a[k] == b[k]).all(), (m.name, k)


def test_tiny_dense_cube_many_events(gpu):
    # dense box, high release rate: bindings, releases, births and compaction every step;
    # ragged sizes (not multiples of any tile), several cells, wall agents
    m = tiny_cube(L=301, n_a=1237, n_b=1111, p_bind=0.7, p_rel=0.05, cell=64)
    run_both(gpu, m, 40, chunks=8)


def test_large_displacements(gpu):
    # sigma = 300 / 250 units: displacements up to +-1100, several cells per step (cell 100)
    A, B, Cx = 0, 1, 2
    m = Model(
        name="bigsigma", species=[Species("A", 1), Species("B", 1),
                                  Species("C", 2, channels=[Channel(CH_RELEASE, prob_to_thr(0.02), A, B)])],
        reactions=[Reaction(A, B, Cx, 2500, prob_to_thr(0.5))],
        compartments=[Compartment(SHAPE_CUBE, L=3000)], table_bits=12, tables=stack_tables([300.0, 250.0], 12),
        extent=(3000,) * 3, seed=21, place_seed=22,
        seed_records=[SeedRecord(A, 4000), SeedRecord(B, 4000)], n_steps=24, cell_size=100).finalize()
    run_both(gpu, m, 24, chunks=3)


def test_cell_size_independence_on_gpu(gpu):
    m = tiny_cube(L=400, n_a=1500, n_b=1500, p_rel=0.02)
    ref = None
    for cell in (50, 53, 64, 97, 100, 256, 333, 400):   # odd sizes exercise the multiply-high cell division
        sim = gpu.Sim(m, cell_size=cell); sim.seed_population(); sim.step(12)
        s = sim.read_agents()
        if ref is None:
            ref = s
        for k in ref:
            assert (ref[k] == s[k]).all(), (cell, k)
    orc = oracle_cls()(m); orc.seed_population(); orc.step(12)
    b = orc.read_agents()
    for k in ref:
        assert (ref[k] == b[k]).all()


def test_w0_full_1000_steps(gpu):
    """[CFG 0] in full: 1,000 steps, every counts row and the final id-sorted state."""
    m = configs.w0(cell_size=512)
    sim, orc = run_both(gpu, m, 1000, chunks=4)
    c = sim.read_counts()[:, 0, :].astype(np.int64)
    assert (c[:, 0] + c[:, 2] == 5000).all() and (c[:, 1] + c[:, 2] == 5000).all()


def test_w1_scaled_cascade(gpu):
    m = configs.w1(scale=0.01, n_steps=300, cell_size=256)     # 10.5 k agents, sphere R = 1.08 um
    run_both(gpu, m, 300, chunks=3)


def test_w2_scaled_replicas(gpu):
    m = configs.w2(scale=0.002, n_steps=200, cell_size=256)    # 8 replicas, ~17.7 k agents
    sim, orc = run_both(gpu, m, 200, chunks=2)
    c = sim.read_counts()
    assert c.shape[1] == 8


def test_w3_scaled_nucleus_expression_delay(gpu):
    m = configs.w3(scale=0.004, n_steps=700, delay=40, cell_size=256)
    ix = {s.name: i for i, s in enumerate(m.species)}
    Oracle = oracle_cls()
    orc = Oracle(m); orc.seed_population()
    a = orc.read_agents()
    genes = np.nonzero(a["species"] == ix["GENE"])[0]
    extra, n0 = 400, len(a["id"])
    rng = np.random.default_rng(1)
    pick = genes[rng.integers(0, 2, extra)]
    pos = {k: np.concatenate([a[k], (a[k][pick] + rng.integers(-60, 60, extra)).astype(np.int32)]) for k in "xyz"}
    sp = np.concatenate([a["species"], np.full(extra, ix["pERK_n"], np.uint16)])
    ids = np.concatenate([a["id"], np.arange(n0, n0 + extra, dtype=np.uint32)])
    sim = gpu.Sim(m)
    for s in (sim, orc):
        s.load_agents(pos["x"], pos["y"], pos["z"], sp, ids)
    for c in range(7):
        sim.step(100); orc.step(100)
        assert_same(sim, orc, f"W3 chunk {c}")
    c = sim.read_counts()[:, 0, :]
    assert orc.info()["t_first0"] != 0xFFFFFFFF
    assert c[-1, ix["F_n"]] + c[-1, ix["GENE:F"]] == 2            # the delayed births happened
    assert c[:, ix["mRNA_n"]].max() + c[:, ix["mRNA_c"]].max() > 0


def test_channel_kinds_and_priority(gpu):
    # BIRTH + DEGRADE + CONVERT + RELEASE on one species, several births per parent per step
    X, Y, Z, W = 0, 1, 2, 3
    sp = [Species("X", 1, channels=[Channel(CH_BIRTH, prob_to_thr(0.2), prod1=Z),
                                    Channel(CH_DEGRADE, prob_to_thr(0.05)),
                                    Channel(CH_BIRTH, prob_to_thr(0.3), prod1=W),
                                    Channel(CH_RELEASE, prob_to_thr(0.1), Y, Z)]),
          Species("Y", 1, channels=[Channel(CH_CONVERT, prob_to_thr(0.1), X)]),
          Species("Z", 2, channels=[Channel(CH_DEGRADE, prob_to_thr(0.3))]),
          Species("W", 0, channels=[Channel(CH_DEGRADE, prob_to_thr(0.5))])]
    m = Model(name="chan", species=sp, reactions=[Reaction(Y, Z, W, 2500, prob_to_thr(0.5))],
              compartments=[Compartment(SHAPE_CUBE, L=700)], table_bits=12,
              tables=stack_tables([44.7214, 31.6228], 12), extent=(700,) * 3, seed=99, place_seed=98,
              seed_records=[SeedRecord(X, 3000), SeedRecord(Y, 777)], n_steps=60, cell_size=64)
    m.capacity = 60000; m.id_capacity = 400000
    m.finalize()
    run_both(gpu, m, 60, chunks=6)


def test_w4_200k_and_step_split(gpu):
    m = configs.w4(n=200_000, n_steps=30)
    sim, orc = run_both(gpu, m, 30, chunks=2)
    # step(a); step(b) == step(a+b) on the GPU, and reload from a dump
    s2 = gpu.Sim(m); s2.seed_population(); s2.step(7); s2.step(23)
    a, b = sim.read_agents(), s2.read_agents()
    for k in a:
        assert (a[k] == b[k]).all()
    s3 = gpu.Sim(m); s3.seed_population(); s3.step(7)
    d = s3.read_agents(); inf = s3.info()
    perm = np.random.default_rng(0).permutation(len(d["id"]))     # memory order must not matter
    s4 = gpu.Sim(m)
    s4.load_agents(*(d[k][perm] for k in ("x", "y", "z", "species", "id")), step=7, next_id=inf["next_id"])
    s4.step(23)
    c = s4.read_agents()
    for k in a:
        assert (a[k] == c[k]).all()


def test_large_capacity_kernel_configuration(gpu):
    """K1/K3 are instantiated with more agents per thread from a capacity of 2 M agents on (MoveCfgLarge);
    the same small populations must give the same result through that instantiation (ragged tiles, a sphere
    with membrane crossings, and a cube)."""
    m = configs.w4(n=150_003, n_steps=12)
    m.capacity = 2_100_000
    m.finalize()
    run_both(gpu, m, 12, chunks=2)
    m = configs.w3(scale=0.004, n_steps=60)
    m.capacity = 2_100_000
    m.finalize()
    run_both(gpu, m, 60, chunks=2)


def test_crowded_single_cell(gpu):
    """70,000 non-binding agents in ONE cell (ranks far beyond 16 bits, one histogram counter taking every
    atomic); a second pair of species keeps a few bindings going in the same cell."""
    X, A, B, Cx = 0, 1, 2, 3
    m = Model(name="crowded", species=[Species("X", 1), Species("A", 1), Species("B", 1), Species("C", 2)],
              reactions=[Reaction(A, B, Cx, 2500, prob_to_thr(0.5))],
              compartments=[Compartment(SHAPE_CUBE, L=3000)], table_bits=12,
              tables=stack_tables([44.7214, 31.6228], 12), extent=(3000,) * 3, seed=5, place_seed=6,
              seed_records=[SeedRecord(X, 70_000), SeedRecord(A, 300), SeedRecord(B, 300)], n_steps=3, cell_size=4096)
    m.finalize()
    run_both(gpu, m, 3, chunks=1)


def test_w4_1m_full_size_steps(gpu):
    """[CFG 4] N = 1 M in the bench launch configuration, 6 steps, full state compare."""
    m = configs.w4(n=1_000_000, n_steps=6)
    run_both(gpu, m, 6, chunks=2)


@pytest.mark.slow
def test_w4_16m_full_size_two_steps(gpu):
    """[CFG 4] N = 16 M (the bench workload): 2 steps, every agent compared with the oracle."""
    m = configs.w4(n=16_000_000, n_steps=2)
    run_both(gpu, m, 2, chunks=1)


def test_w1_full_size_steps(gpu):
    """[CFG 1] at full size (1.05 M agents, sphere R = 5 um) in the bench launch configuration."""
    m = configs.w1(n_steps=4)
    run_both(gpu, m, 4, chunks=2)


def test_w3_full_size_steps(gpu):
    """[CFG 3] at full size (337,502 agents, shell + nucleus, membrane crossings)."""
    m = configs.w3(n_steps=24)
    run_both(gpu, m, 24, chunks=2)


@pytest.mark.slow
def test_w2_full_size_two_steps(gpu):
    """[CFG 2] at full size: 8 replicas, 8,854,860 agents, every agent compared with the oracle."""
    m = configs.w2(n_steps=2)
    run_both(gpu, m, 2, chunks=1)


def test_concurrent_handles_on_separate_streams(gpu):
    """independent seeds run concurrently, one handle + one CUDA stream each; every one of
    them must still match its own oracle run bit for bit."""
    import torch

    models = []
    for r in range(4):
        m = tiny_cube(L=300 + 7 * r, n_a=900 + 50 * r, n_b=800, p_rel=0.03, seed=40 + r)
        models.append(m)
    sims = [gpu.Sim(m, stream=torch.cuda.Stream()) for m in models]
    for s in sims:
        s.seed_population()
    for _ in range(3):                       # interleaved asynchronous stepping on four streams
        for s in sims:
            s.step_async(9)
    for s, m in zip(sims, models):
        s.step(0)
        orc = oracle_cls()(m); orc.seed_population(); orc.step(27)
        assert_same(s, orc, m.name)


def test_empty_population_and_mid_run_seeding(gpu):
    """Degenerate cases: stepping an empty handle, then adding agents mid-run (run-time treatment
    change) with fresh ids, twice, against the oracle doing the same."""
    m = tiny_cube(L=320, n_a=700, n_b=650, p_rel=0.02, seed=77)
    sim = gpu.Sim(m); orc = oracle_cls()(m)
    sim.step(3); orc.step(3)                               # nothing there yet
    assert_same(sim, orc, "empty")
    assert sim.info()["n_live"] == 0
    sim.seed_population(); orc.seed_population()
    sim.step(9); orc.step(9)
    assert_same(sim, orc, "after first seeding")
    extra = [SeedRecord(1, 333), SeedRecord(0, 17)]        # a dose of B and a few A, placed from another seed
    sim.seed_population(extra, place_seed=1234); orc.seed_population(extra, place_seed=1234)
    assert_same(sim, orc, "right after the mid-run dose")
    sim.step(11); orc.step(11)
    assert_same(sim, orc, "after the mid-run dose")


def test_errors(gpu):
    from paper_2606_14603_b200.binding import E_CAPACITY, E_INVAL, SimError

    m = tiny_cube()
    m.cell_size = 49
    with pytest.raises(SimError) as e:
        gpu.Sim(m)
    assert e.value.code == E_INVAL
    m = tiny_cube(p_bind=0.0, p_rel=1.0)
    m.capacity = 2100
    sim = gpu.Sim(m)
    n = 2000
    pos = np.random.default_rng(1).integers(0, 400, size=(3, n)).astype(np.int32)
    sim.load_agents(pos[0], pos[1], pos[2], np.full(n, 2, np.uint16), np.arange(n, dtype=np.uint32))
    with pytest.raises(SimError) as e:      # every C releases a newborn: 4,000 > capacity
        sim.step(1)
    assert e.value.code == E_CAPACITY
    # agent data handed to sim_load_agents is validated on the device; the handle stays usable
    m = tiny_cube()
    sim = gpu.Sim(m)
    ok = np.arange(10, dtype=np.uint32)
    xs = np.full(10, 5, np.int32)
    for bad in ({"species": np.full(10, 7, np.uint16)}, {"id": ok + 100}, {"x": np.full(10, -3, np.int32)}):
        a = {"x": xs, "y": xs, "z": xs, "species": np.zeros(10, np.uint16), "id": ok}
        a.update(bad)
        with pytest.raises(SimError) as e:
            sim.load_agents(a["x"], a["y"], a["z"], a["species"], a["id"], next_id=10)
        assert e.value.code == E_INVAL
        assert sim.info()["n_live"] == 0
    sim.load_agents(xs, xs, xs, np.zeros(10, np.uint16), ok, next_id=10)
    sim.step(2)
    assert sim.info()["n_live"] == 10
    m = tiny_cube(); m.counts_rows = 4
    sim = gpu.Sim(m); sim.seed_population(); sim.step(3)
    with pytest.raises(SimError):
        sim.step(1)
