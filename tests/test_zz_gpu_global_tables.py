"""GPU parity for the one kernel configuration no other test reaches: Gaussian displacement tables too large for shared
memory (> 160 KB: 16-bit tables, or many sigma classes), where K3 / K5 / the prologue / the move hook are the
`kGaussSmem = false` instantiations that read the tables from global memory.  Found by line coverage of the emulation
build (tests/test_simt_kernels.py), which runs the same body on the CPU; this file was added while the GPU pool was
closed to the repository, so it is collected last: a failure here cannot hide another GPU test behind `pytest -x`."""
import numpy as np
import pytest

from workloads.model import (CH_BIRTH, CH_CONVERT, CH_DEGRADE, CH_DELAYED_BIRTH, CH_RELEASE, SHAPE_CUBE, SHAPE_SPHERE,
                             Channel, Compartment, Model, Reaction, SeedRecord, Species, prob_to_thr, stack_tables)


@pytest.fixture(scope="module")
def gpu():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_14603_b200 as pkg

    pkg.load_library()
    return pkg


def big_table_models():
    A, B, Cx = 0, 1, 2
    sp = [Species("A", 1), Species("B", 2), Species("C", 3, channels=[Channel(CH_RELEASE, prob_to_thr(0.03), A, B)])]
    rx = [Reaction(A, B, Cx, 2500, prob_to_thr(0.6))]
    # 4 rows x 2^16 entries x 2 B = 512 KB of tables
    cube = Model(name="tables16_cube", species=sp, reactions=rx, compartments=[Compartment(SHAPE_CUBE, L=450)],
                 table_bits=16, tables=stack_tables([44.7214, 31.6228, 20.0], 16), extent=(450,) * 3, seed=31,
                 place_seed=32, seed_records=[SeedRecord(A, 2100), SeedRecord(B, 1900)], n_steps=30, cell_size=64).finalize()
    # 24 sigma classes x 2^12 entries x 2 B = 196 KB, in a sphere (no-flux wall)
    sig = [10.0 + 3.0 * k for k in range(23)]
    sp2 = [Species("A", 23), Species("B", 7), Species("C", 1, channels=[Channel(CH_RELEASE, prob_to_thr(0.03), A, B)])]
    R = 400
    sphere = Model(name="tables24_sphere", species=sp2, reactions=rx,
                   compartments=[Compartment(SHAPE_SPHERE, cx=R, cy=R, cz=R, r_out=R, r_in=-1)], table_bits=12,
                   tables=stack_tables(sig, 12), extent=(2 * R + 1,) * 3, seed=33, place_seed=34,
                   seed_records=[SeedRecord(A, 2500), SeedRecord(B, 2500)], n_steps=30, cell_size=100).finalize()
    return cube, sphere


def body_large_gaussian_tables(gpu):
    from test_gpu_parity import oracle_cls, run_both

    for m in big_table_models():
        assert m.tables.nbytes > 160 * 1024
        run_both(gpu, m, 30, chunks=3)
        sim = gpu.Sim(m); orc = oracle_cls()(m)              # the move-only hook has its own instantiation
        sim.seed_population(); orc.seed_population()
        sim.debug_move_only(); orc.debug_move_only()
        a, b = sim.read_agents(), orc.read_agents()
        for k in ("id", "species", "x", "y", "z"):
            assert (a[k] == b[k]).all(), (m.name, k)


def maximum_size_model():
    """Every table at its maximum (include/molsim.h): 64 species in 8 compartments (four shells with their cores,
    membrane twins across each), 64 reactions, 8 t_first rules with marked and delayed births, 4 channels on many species,
    64 replicas, 255 sigma classes would not fit a test: 31 are used."""
    rng = np.random.default_rng(64)
    R, r_in = 150, 80
    comps = []
    for k in range(4):                      # four concentric shell + core pairs side by side along y
        cy = R + k * (2 * R + 40)
        comps += [Compartment(SHAPE_SPHERE, R, cy, R, r_out=R, r_in=r_in), Compartment(SHAPE_SPHERE, R, cy, R, r_out=r_in)]
    n_sp, n_cls = 64, 31
    species = [Species(f"S{i}", sigma_class=1 + i % n_cls, compartment=i % 8) for i in range(n_sp)]
    by_comp = {c: [i for i in range(n_sp) if i % 8 == c] for c in range(8)}
    for i in range(0, n_sp, 2):             # twins: shell species i <-> core species i + 1 of the same pair
        species[i].cross_to, species[i].cross_thr = i + 1, prob_to_thr(0.3)
        species[i + 1].cross_to, species[i + 1].cross_thr = i, 0xFFFFFFFF
    reactions, seen = [], set()
    while len(reactions) < 64:
        c = int(rng.integers(8))
        a, b, cx = (int(v) for v in rng.choice(by_comp[c], 3))
        if (min(a, b), max(a, b)) in seen:
            continue
        seen.add((min(a, b), max(a, b)))
        r = int(rng.integers(10, 41))
        reactions.append(Reaction(a, b, cx, r * r, prob_to_thr(float(rng.uniform(0.2, 1.0)))))
    reactions[0].r2 = 40 * 40
    for rule in range(8):                   # one marked birth + one delayed birth per rule
        s = species[rule * 8]
        mine = by_comp[s.compartment]
        s.channels = [Channel(CH_BIRTH, prob_to_thr(0.01), prod1=int(mine[1]), rule=rule, marks_first=True),
                      Channel(CH_DELAYED_BIRTH, 2 + rule % 3, prod1=int(mine[2]), rule=rule),
                      Channel(CH_RELEASE, prob_to_thr(0.02), int(mine[3]), int(mine[4])),
                      Channel(CH_DEGRADE, prob_to_thr(0.005))]
    for i in range(1, n_sp, 3):
        mine = by_comp[species[i].compartment]
        species[i].channels = [Channel(CH_CONVERT, prob_to_thr(0.02), int(mine[5])),
                               Channel(CH_RELEASE, prob_to_thr(0.03), int(mine[6]), int(mine[7]))]
    n_rep, shift = 64, 9                    # tile 512 >= 2 R + 1 + R_max + 1
    recs = [SeedRecord(int(rng.integers(n_sp)), int(rng.integers(20, 60)), rep) for rep in range(n_rep) for _ in range(3)]
    ext_y = comps[-1].cy + R + 1
    m = Model(name="maximum_sizes", species=species, reactions=reactions, compartments=comps, table_bits=8,
              tables=stack_tables([3.0 + 0.5 * k for k in range(n_cls)], 8), extent=(n_rep << shift, ext_y, 2 * R + 1),
              seed=640, place_seed=641, seed_records=recs, n_steps=16, cell_size=40, n_replicas=n_rep, stride_shift=shift,
              n_rules=8)
    m.capacity = 4 * m.n_agents0 + 4096
    return m.finalize()


def body_maximum_table_sizes(gpu):
    from paper_2606_14603_b200.binding import check_config
    from test_gpu_parity import run_both

    m = maximum_size_model()
    assert check_config(m) is None, check_config(m)
    assert (len(m.species), len(m.reactions), len(m.compartments), m.n_replicas, m.n_rules) == (64, 64, 8, 64, 8)
    sim, orc = run_both(gpu, m, 16, chunks=4)
    c = orc.read_counts()
    assert c.shape[1:] == (64, 64) and (c[-1].sum(axis=1) > 0).all()          # every replica is populated
    assert (orc.read_t_first() != 0xFFFFFFFF).any()                            # marked births happened


@pytest.mark.gpu
def test_maximum_table_sizes(gpu):
    body_maximum_table_sizes(gpu)


@pytest.mark.gpu
def test_large_gaussian_tables_in_global_memory(gpu):
    body_large_gaussian_tables(gpu)


@pytest.mark.gpu
def test_random_models_parity(gpu):
    """Parity fuzzing: 60 seeded random models (tests/random_models.py: cubes, spheres, shell + nucleus with membrane twins,
    replicas; random species, sigma classes, reactions up to R = cell size, every channel kind) stepped on the GPU and on
    the oracle; full state, counts, info and checksum compared.  The CPU tier runs the same body on the emulation."""
    from paper_2606_14603_b200.binding import check_config
    from random_models import fuzz_parity
    from test_gpu_parity import assert_same, oracle_cls

    assert fuzz_parity(gpu, range(1000, 1060), check_config, oracle_cls(), assert_same) >= 50


@pytest.mark.gpu
def test_random_api_sequences_parity(gpu):
    """Random sequences of step(n) / mid-run seeding / checkpoint reload in permuted order / per-kernel profiling on and
    off, applied to the GPU handle and to the oracle alike, full state compared after every call: the host-side state
    machine (histogram validity, ping-pong parity, 1-step and 8-step graphs, direct launches)."""
    from paper_2606_14603_b200.binding import check_config
    from random_models import api_sequence_parity
    from test_gpu_parity import assert_same, oracle_cls

    assert api_sequence_parity(gpu, range(2000, 2030), check_config, oracle_cls(), assert_same) >= 25


def body_degenerate_populations(gpu):
    """Degenerate populations: exactly `capacity` agents (the last tile of every pass ends at the last slot, K4's bulk
    copies and group reads run into the slack behind it), a population in which everybody degrades in the first step
    (stepping goes on with nobody alive), and a single agent."""
    from test_gpu_parity import run_both, tiny_cube

    m = tiny_cube(L=300, n_a=1024, n_b=1024, p_bind=0.6, p_rel=0.0, cell=64)       # no release: the population only shrinks
    m.capacity = 2048
    run_both(gpu, m, 6, chunks=2)
    X = 0
    m = Model(name="all_degrade", species=[Species("X", 1, channels=[Channel(CH_DEGRADE, 0xFFFFFFFF)])], reactions=[],
              compartments=[Compartment(SHAPE_CUBE, L=500)], table_bits=10, tables=stack_tables([30.0], 10),
              extent=(500,) * 3, seed=5, place_seed=6, seed_records=[SeedRecord(X, 3000)], n_steps=5, cell_size=50).finalize()
    sim, orc = run_both(gpu, m, 5, chunks=5)
    assert sim.info()["n_live"] == 0 and sim.read_counts()[1:].sum() == 0
    m = tiny_cube(L=300, n_a=1, n_b=0, cell=64)
    m.seed_records = [r for r in m.seed_records if r.count]
    run_both(gpu, m, 9, chunks=3)


@pytest.mark.gpu
def test_degenerate_populations(gpu):
    body_degenerate_populations(gpu)
