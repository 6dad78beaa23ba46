"""Seeded random models for parity fuzzing (an input generator: it holds none of the step's arithmetic).

`random_model(seed)` draws a valid model of a random shape — a cube, a sphere, a shell around a nucleus with membrane
twins, or several replicas of a sphere — with a random number of species and sigma classes, random bimolecular reactions
(homodimers included, radii from a few units up to exactly the cell size, thresholds from never to always), random
unimolecular channels of every kind (BIRTH, marked BIRTH + DELAYED_BIRTH, RELEASE, CONVERT, DEGRADE, several per
species), random table resolution, cell size and population (a few hundred to 16,000 agents; volumes from one cell to
several hundred).  The draws respect the validation rules V1-V7 of include/molsim.h; the callers check that with
`sim_check_config` and skip the rare draw that does not."""
import numpy as np

from workloads.model import (CH_BIRTH, CH_CONVERT, CH_DEGRADE, CH_DELAYED_BIRTH, CH_RELEASE, NONE16, SHAPE_CUBE,
                             SHAPE_SPHERE, Channel, Compartment, Model, Reaction, SeedRecord, Species, prob_to_thr,
                             stack_tables)


def random_model(seed: int, n_agents=(600, 3500), steps=(6, 12), allow_big=True) -> Model:
    rng = np.random.default_rng(seed)
    pick = lambda seq: seq[int(rng.integers(len(seq)))]                                      # noqa: E731
    shape = pick(["cube", "cube", "sphere", "nucleus", "replicas"])
    table_bits = int(rng.integers(6, 13))
    n_classes = int(rng.integers(1, 5))
    # radii and cell size: R_max anywhere from a few units to exactly the cell edge
    cell = int(pick([16, 23, 40, 64, 100, 128]))
    r_max = int(pick([cell, cell, max(3, cell // 2), max(3, cell // 3), cell - 1]))
    size = int(rng.integers(4, 9)) * cell + int(rng.integers(0, cell))      # not a multiple of the cell edge
    crowd = rng.random()
    if crowd < 0.15:                                                         # one or two cells per axis: everybody is a neighbour
        size = int(rng.integers(cell // 2 + 8, 2 * cell))
    elif crowd < 0.25 and allow_big:                                         # many tiles per block: the K4 ring wraps around
        n_agents = (8000, 16000)
    sig_hi = min(size / 7.0, 2.5 * cell)
    sigmas = [float(rng.uniform(2.0, sig_hi)) for _ in range(n_classes)]
    n_replicas, stride_shift = 1, 31
    if shape == "cube":
        comps = [Compartment(SHAPE_CUBE, L=size)]
        extent = (size,) * 3
    else:
        R = size // 2
        if shape == "nucleus":
            r_in = int(R * rng.uniform(0.35, 0.7))
            comps = [Compartment(SHAPE_SPHERE, R, R, R, r_out=R, r_in=r_in), Compartment(SHAPE_SPHERE, R, R, R, r_out=r_in)]
        else:
            comps = [Compartment(SHAPE_SPHERE, R, R, R, r_out=R)]
        extent = (2 * R + 1,) * 3
        if shape == "replicas":
            n_replicas = int(rng.integers(2, 6))
            stride_shift = int(np.ceil(np.log2(2 * R + 1 + r_max + 1))) + int(rng.integers(0, 2))
            extent = (n_replicas << stride_shift, 2 * R + 1, 2 * R + 1)
    n_comp = len(comps)
    # species: a few per compartment; membrane twins in the nucleus shape
    n_sp = int(rng.integers(3, 11))
    species = [Species(f"S{i}", sigma_class=int(rng.integers(0 if rng.random() < 0.15 else 1, n_classes + 1)),
                       compartment=int(rng.integers(n_comp)) if i >= n_comp else i) for i in range(n_sp)]
    if shape == "nucleus":
        for _ in range(int(rng.integers(1, 4))):
            a = int(rng.integers(n_sp))
            others = [j for j in range(n_sp) if species[j].compartment != species[a].compartment]
            if others and species[a].sigma_class:
                species[a].cross_to = int(pick(others))
                species[a].cross_thr = int(pick([prob_to_thr(0.05), prob_to_thr(0.5), 0xFFFFFFFF]))
    by_comp = {c: [i for i in range(n_sp) if species[i].compartment == c] for c in range(n_comp)}
    # reactions within a compartment, homodimers included, no unordered pair twice
    reactions, seen = [], set()
    for _ in range(int(rng.integers(1, 6))):
        c = int(rng.integers(n_comp))
        a, b, cx = int(pick(by_comp[c])), int(pick(by_comp[c])), int(pick(by_comp[c]))
        if (min(a, b), max(a, b)) in seen:
            continue
        seen.add((min(a, b), max(a, b)))
        r = int(pick([r_max, r_max, max(2, r_max // 2), int(rng.integers(2, r_max + 1))]))
        reactions.append(Reaction(a, b, cx, r * r, int(pick([0, prob_to_thr(0.1), prob_to_thr(0.5), prob_to_thr(0.9), 0xFFFFFFFF]))))
    if reactions:       # one of them has the largest radius the cell admits
        reactions[0].r2 = r_max * r_max
    # unimolecular channels
    n_rules = 0
    for i, s in enumerate(species):
        if rng.random() < 0.55:
            continue
        mine = by_comp[s.compartment]
        for _ in range(int(rng.integers(1, 5))):
            kind = int(pick([CH_BIRTH, CH_RELEASE, CH_RELEASE, CH_CONVERT, CH_DEGRADE, CH_DELAYED_BIRTH]))
            p = float(pick([0.002, 0.02, 0.1]))
            if kind == CH_BIRTH:
                marks = n_rules < 8 and rng.random() < 0.4
                s.channels.append(Channel(CH_BIRTH, prob_to_thr(min(p, 0.03)), prod1=int(pick(mine)), rule=n_rules if marks else 0,
                                          marks_first=bool(marks)))
                n_rules += int(marks)
            elif kind == CH_DELAYED_BIRTH:
                if n_rules == 0:
                    continue
                s.channels.append(Channel(CH_DELAYED_BIRTH, int(rng.integers(1, 5)), prod1=int(pick(mine)),
                                          rule=int(rng.integers(n_rules))))
            elif kind == CH_RELEASE:
                s.channels.append(Channel(CH_RELEASE, prob_to_thr(p), int(pick(mine)), int(pick(mine))))
            elif kind == CH_CONVERT:
                s.channels.append(Channel(CH_CONVERT, prob_to_thr(p), int(pick(mine))))
            else:
                s.channels.append(Channel(CH_DEGRADE, prob_to_thr(p)))
    # population
    n0 = int(rng.integers(*n_agents))
    recs = []
    weights = rng.dirichlet(np.ones(n_sp))
    for rep in range(n_replicas):
        for i in range(n_sp):
            k = int(round(n0 * weights[i] / n_replicas))
            if k and rng.random() < 0.9:
                recs.append(SeedRecord(i, k, rep))
    n_steps = int(rng.integers(*steps))
    m = Model(name=f"random{seed}_{shape}", species=species, reactions=reactions, compartments=comps, table_bits=table_bits,
              tables=stack_tables(sigmas, table_bits), extent=extent, seed=int(rng.integers(1, 2**62)),
              place_seed=int(rng.integers(1, 2**62)), seed_records=recs, n_steps=n_steps, cell_size=cell,
              n_replicas=n_replicas, stride_shift=stride_shift, n_rules=max(1, n_rules))
    m.capacity = 6 * max(n0, 1) + 4096
    m.id_capacity = 12 * max(n0, 1) + 65536
    return m.finalize()


def fuzz_parity(pkg, seeds, check_config, oracle_cls, assert_same):
    """Steps every valid random model on `pkg.Sim` and on the oracle; full state, counts and info compared after seeding,
    half way and at the end.  Returns the number of models run."""
    ran = 0
    for seed in seeds:
        m = random_model(seed)
        if check_config(m) is not None or not m.seed_records:
            continue
        sim, orc = pkg.Sim(m), oracle_cls(m)
        sim.seed_population(); orc.seed_population()
        assert_same(sim, orc, f"{m.name} seeding")
        half = m.n_steps // 2
        for n in (half, m.n_steps - half):
            sim.step(n); orc.step(n)
            assert_same(sim, orc, f"{m.name} after {n} more steps")
        if hasattr(sim, "read_checksum"):
            assert sim.read_checksum() == orc.read_checksum(), m.name
        ran += 1
    return ran


def api_sequence_parity(pkg, seeds, check_config, oracle_cls, assert_same, n_ops=14):
    """Random sequences of API calls — step(n) with n from 0 to 19 (mixes the 8-step and 1-step graphs and both parities of
    the ping-pong), mid-run seeding, a checkpoint written back in permuted order (sim_load_agents + t_first), per-kernel
    profiling switched on and off (direct launches instead of graph replay) — applied to `pkg.Sim` and to the oracle
    alike; the full state is compared after every call.  This exercises the host-side state machine of the library
    (histogram validity, buffer parity, graph selection), not new arithmetic."""
    ran = 0
    for seed in seeds:
        rng = np.random.default_rng(10_000 + seed)
        m = random_model(seed, n_agents=(400, 1500), steps=(6, 7), allow_big=False)
        m.counts_rows = 400
        m.capacity *= 2
        if check_config(m) is not None or not m.seed_records:
            continue
        sim, orc = pkg.Sim(m), oracle_cls(m)
        if rng.random() < 0.7:
            sim.seed_population(); orc.seed_population()
        for k in range(n_ops):
            op = rng.choice(["step", "step", "step", "seed", "reload", "profile", "checksum"])
            if op == "step":
                n = int(rng.choice([0, 1, 2, 3, 7, 8, 9, 16, 19]))
                if sim.info()["step"] + n >= m.counts_rows - 1:
                    continue
                errs = []
                for s in (sim, orc):
                    try:
                        s.step(n)
                        errs.append(0)
                    except RuntimeError as e:            # a population that outgrows its slots or ids: both sides must say so,
                        errs.append(getattr(e, "code", None))     # on the same call, with the same code
                assert errs[0] == errs[1], (m.name, k, errs)
                if errs[0]:
                    break
            elif op == "seed":
                recs = [r for r in m.seed_records if rng.random() < 0.3][:3]
                recs = [type(r)(r.species, max(1, r.count // 10), r.replica) for r in recs]
                place = int(rng.integers(1, 2**40))
                sim.seed_population(recs, place_seed=place); orc.seed_population(recs, place_seed=place)
            elif op == "reload":
                a, info, tf = sim.read_agents(), sim.info(), sim.read_t_first()
                perm = rng.permutation(len(a["id"]))
                for s in (sim, orc):
                    s.load_agents(*(a[f][perm] for f in ("x", "y", "z", "species", "id")), step=info["step"],
                                  next_id=info["next_id"])
                    s.load_t_first(tf)
            elif op == "profile":
                sim.profile_enable(bool(rng.integers(2)))
            else:
                assert sim.read_checksum() == orc.read_checksum(), (m.name, k)
            assert_same(sim, orc, f"{m.name} op {k} ({op})")
        ran += 1
    return ran
