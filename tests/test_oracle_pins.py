"""Pins of the CPU oracle against what the model and the mathematics fix (CPU only).

Each test names the DESIGN.md reading / BASELINE.json north_star clause it pins.  None of
these touches the CUDA path.
"""
import numpy as np
import pytest
from scipy.spatial import cKDTree

from oracle.binding import (E_INVAL, MODE_BRUTE, MODE_GRID, NOPROP, Oracle,
                            OracleError, philox)
from workloads import configs, model
from workloads.model import (CH_DEGRADE, CH_RELEASE, SHAPE_CUBE, SHAPE_SPHERE,
                             Channel, Compartment, Model, Reaction, SeedRecord,
                             Species, prob_to_thr, stack_tables)


# --------------------------------------------------------------------------- Philox (S2)
def test_philox_matches_torch_cpu_engine(torch_philox):
    rng = np.random.default_rng(123)
    ctr = rng.integers(0, 2**32, size=(20000, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(20000, 2), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0; key[0] = 0
    ctr[1] = 0xFFFFFFFF; key[1] = 0xFFFFFFFF
    ref = torch_philox(ctr, key)
    for i in range(len(ctr)):
        assert (philox(ctr[i], key[i]) == ref[i]).all(), i


def test_philox_is_injective_in_counter():
    outs = {tuple(philox([i, 0, 7, 1], [5, 0])) for i in range(4096)}
    assert len(outs) == 4096
    assert tuple(philox([1, 0, 7, 1], [5, 0])) != tuple(philox([1, 0, 7, 1], [6, 0]))


# --------------------------------------------------------------------------- helpers
def tiny_cube(L=400, n_a=1000, n_b=1000, p_bind=0.5, p_rel=1e-3, cell=64, seed=11, sig=(44.7214, 31.6228)):
    A, B, Cx = 0, 1, 2
    m = Model(
        name="tiny", species=[Species("A", 1), Species("B", 1),
                              Species("C", 2, channels=[Channel(CH_RELEASE, prob_to_thr(p_rel), A, B)])],
        reactions=[Reaction(A, B, Cx, 2500, prob_to_thr(p_bind))],
        compartments=[Compartment(SHAPE_CUBE, L=L)], table_bits=12, tables=stack_tables(list(sig), 12),
        extent=(L, L, L), seed=seed, place_seed=seed,
        seed_records=[SeedRecord(A, n_a), SeedRecord(B, n_b)], n_steps=64, cell_size=cell)
    return m.finalize()


def state_equal(a, b):
    return all((a[k] == b[k]).all() and len(a[k]) == len(b[k]) for k in ("x", "y", "z", "species", "id"))


# --------------------------------------------------------------------------- seeding (S15)
def test_seeding_uniform_and_ids():
    m = configs.w0()
    o = Oracle(m); o.seed_population()
    a = o.read_agents()
    assert (a["id"] == np.arange(10000)).all()
    assert (a["species"][:5000] == 0).all() and (a["species"][5000:] == 1).all()
    for k in "xyz":
        assert a[k].min() >= 0 and a[k].max() < 10000
        h, _ = np.histogram(a[k], bins=10, range=(0, 10000))
        chi2 = ((h - 1000.0) ** 2 / 1000.0).sum()
        assert chi2 < 35.0          # 9 dof, p ~ 1e-4
    c = o.read_counts()
    assert c.shape == (1, 1, 3) and list(c[0, 0]) == [5000, 5000, 0]


def test_seeding_sphere_shell_valid_and_radial_law():
    m = configs.w3(scale=0.05)
    o = Oracle(m); o.seed_population()
    a = o.read_agents()
    R = m.compartments[0].r_out; Rn = m.compartments[1].r_out
    r2 = sum((a[k].astype(np.int64) - R) ** 2 for k in "xyz")
    comp = np.array([s.compartment for s in m.species])[a["species"]]
    assert ((r2[comp == 0] > Rn * Rn) & (r2[comp == 0] <= R * R)).all()
    assert (r2[comp == 1] <= Rn * Rn).all()
    # uniform in the shell: fraction with r < r_mid equals the volume fraction
    r = np.sqrt(r2[comp == 0].astype(np.float64))
    rm = 0.8 * R
    frac = (r < rm).mean(); exp = (rm**3 - Rn**3) / (R**3 - Rn**3)
    assert abs(frac - exp) < 4 * np.sqrt(exp * (1 - exp) / len(r))


# --------------------------------------------------------------------------- move (S2,S3,S5)
def test_move_matches_independent_rng_and_mirror(torch_philox):
    """x' = mirror(x + table[r_a >> (32-B)]) with r = Philox(key=seed; ctr=(id,0,t,1)), words x,y,z."""
    m = tiny_cube(L=400, n_a=500, n_b=500, seed=0x1234567855AA)
    o = Oracle(m); o.seed_population()
    before = o.read_agents()
    o.debug_move_only()
    after = o.read_agents()
    ids = before["id"].astype(np.uint32)
    ctr = np.stack([ids, np.zeros_like(ids), np.zeros_like(ids), np.ones_like(ids)], axis=1)
    r = torch_philox(ctr, [m.seed & 0xFFFFFFFF, m.seed >> 32])
    tab = m.tables[1].astype(np.int64)       # A and B share sigma class 1
    L = 400
    hit_wall = 0
    for axis, k in enumerate("xyz"):
        q = before[k].astype(np.int64) + tab[r[:, axis] >> 20]
        hit_wall += int(((q < 0) | (q >= L)).sum())
        q = np.where(q < 0, -1 - q, q)
        q = np.where(q >= L, 2 * L - 1 - q, q)
        assert (after[k] == q).all()
    assert hit_wall > 50          # the mirror branch was exercised


def test_mirror_unit_cases_via_wall_agents(torch_philox):
    # agents sitting on the walls: q = -1 -> 0, q = -2 -> 1, q = L -> L-1 (S5) all occur and stay in [0, L)
    m = tiny_cube(L=400, seed=9)
    o = Oracle(m)
    n = 2000
    x = np.where(np.arange(n) % 2 == 0, 0, 399).astype(np.int32)
    o.load_agents(x, x, x, np.zeros(n, np.uint16), np.arange(n, dtype=np.uint32))
    o.debug_move_only()
    a = o.read_agents()
    for k in "xyz":
        assert a[k].min() >= 0 and a[k].max() < 400


def test_free_diffusion_msd_closed_form():
    """E[dx^2] after n steps = n * var(table) (== 2 D t per axis; MSD = 6 D t), far from walls."""
    L = 20_000
    m = tiny_cube(L=L, n_a=1, n_b=1, cell=512)
    m.capacity = 30000; m.id_capacity = 30000
    o = Oracle(m)
    n = 20000
    p0 = np.random.default_rng(2).integers(5000, 15000, size=(3, n)).astype(np.int32)
    o.load_agents(p0[0], p0[1], p0[2], np.zeros(n, np.uint16), np.arange(n, dtype=np.uint32))
    steps = 25
    o.step(steps)
    a = o.read_agents()
    var_tab = float((m.tables[1].astype(np.float64) ** 2).mean())
    for ax, k in enumerate("xyz"):
        d = a[k].astype(np.float64) - p0[ax]
        assert abs(d.mean()) < 5 * np.sqrt(steps * var_tab / n)
        rel = (d * d).mean() / (steps * var_tab) - 1.0
        assert abs(rel) < 4 * np.sqrt(2.0 / n)
    # sigma^2 = 2 D dt with D = 10 um^2/s, dt = 1 us -> 2000 units^2 per axis per step
    assert abs(var_tab / 2000.0 - 1.0) < 2e-3


def test_cube_uniform_measure_preserved():
    m = tiny_cube(L=300, n_a=4000, n_b=0, p_bind=0.0)
    m.seed_records = [SeedRecord(0, 4000)]
    o = Oracle(m); o.seed_population(); o.step(60)
    a = o.read_agents()
    for k in "xyz":
        h, _ = np.histogram(a[k], bins=6, range=(0, 300))
        exp = 4000 / 6
        assert ((h - exp) ** 2 / exp).sum() < 30.0      # 5 dof


# --------------------------------------------------------------------------- sphere / membrane (S6,S7)
def crossing_model(R=1500, Rn=1000, n=12000, p=0.05, seed=21):
    Xc, Xn = 0, 1
    thr = prob_to_thr(p)
    sp = [Species("X_c", 1, 0, cross_to=Xn, cross_thr=thr), Species("X_n", 1, 1, cross_to=Xc, cross_thr=thr)]
    m = Model(name="cross", species=sp, reactions=[],
              compartments=[Compartment(SHAPE_SPHERE, R, R, R, r_out=R, r_in=Rn),
                            Compartment(SHAPE_SPHERE, R, R, R, r_out=Rn)],
              table_bits=12, tables=stack_tables([89.4427], 12), extent=(2 * R + 1,) * 3,
              seed=seed, place_seed=seed, seed_records=[SeedRecord(Xc, n)], n_steps=4000, cell_size=256)
    return m.finalize()


def test_membrane_compartment_invariant_and_volume_ratio():
    m = crossing_model()
    R, Rn = 1500, 1000
    o = Oracle(m); o.seed_population()
    for _ in range(8):
        o.step(300)
        a = o.read_agents()
        r2 = sum((a[k].astype(np.int64) - R) ** 2 for k in "xyz")
        cyt = a["species"] == 0
        assert ((r2[cyt] > Rn * Rn) & (r2[cyt] <= R * R)).all()     # exact invariant, every agent
        assert (r2[~cyt] <= Rn * Rn).all()
    c = o.read_counts()[:, 0, :].astype(np.float64)
    frac_n = c[1400:, 1].mean() / 12000.0
    exp = Rn**3 / R**3                                            # equal p both ways -> volume ratio
    # lattice-point counts differ from continuum volumes by O(1/R); allow 2 %
    assert abs(frac_n - exp) < 0.02
    assert (c.sum(axis=1) == 12000).all()


def test_sphere_no_flux_radial_law():
    m = crossing_model(p=0.0, n=8000)
    o = Oracle(m); o.seed_population(); o.step(200)
    a = o.read_agents()
    assert (a["species"] == 0).all()
    R, Rn = 1500, 1000
    r = np.sqrt(sum((a[k].astype(np.float64) - R) ** 2 for k in "xyz"))
    rm = 1300.0
    frac = (r < rm).mean(); exp = (rm**3 - Rn**3) / (R**3 - Rn**3)
    assert abs(frac - exp) < 4.5 * np.sqrt(exp * (1 - exp) / len(r))


# --------------------------------------------------------------------------- neighbours (S8, north_star)
@pytest.mark.parametrize("cell", [50, 64, 173, 512])
def test_grid_pairs_equal_bruteforce_and_kdtree(cell):
    m = tiny_cube(L=400, n_a=1000, n_b=1000, cell=cell)
    o = Oracle(m); o.seed_population()
    a = o.read_agents()
    pg = o.debug_pairs(MODE_GRID); pb = o.debug_pairs(MODE_BRUTE)
    assert len(pg) > 20 and (pg == pb).all()
    pts = np.stack([a["x"], a["y"], a["z"]], axis=1).astype(np.float64)
    kd = cKDTree(pts).query_pairs(50.0 + 1e-9, output_type="ndarray")      # library routine
    kd = kd[a["species"][kd[:, 0]] != a["species"][kd[:, 1]]]              # only A-B pairs are eligible
    kd = np.sort(a["id"][kd], axis=1)
    kd = kd[np.lexsort((kd[:, 1], kd[:, 0]))]
    assert kd.shape == pg.shape and (kd == pg).all()


def test_proposals_grid_equals_brute_and_are_valid():
    m = tiny_cube(L=1500, n_a=3000, n_b=3000, cell=50, p_bind=0.5)
    o = Oracle(m); o.seed_population(); o.debug_move_only()
    a = o.read_agents()
    pg = o.debug_proposals(MODE_GRID); pb = o.debug_proposals(MODE_BRUTE)
    assert (pg == pb).all()
    has = pg != NOPROP
    assert has.sum() > 50
    # and at a density where most agents have several candidates (argmin over (d2, id) matters)
    md = tiny_cube(L=300, n_a=1200, n_b=1200, cell=50, p_bind=0.5)
    od = Oracle(md); od.seed_population(); od.debug_move_only()
    assert (od.debug_proposals(MODE_GRID) == od.debug_proposals(MODE_BRUTE)).all()
    pos = np.stack([a["x"], a["y"], a["z"]], axis=1).astype(np.int64)
    idx = {int(i): k for k, i in enumerate(a["id"])}
    pairs = {(int(x), int(y)) for x, y in o.debug_pairs(MODE_BRUTE)}
    n_in_pair = {}
    for x, y in pairs:
        n_in_pair[x] = n_in_pair.get(x, 0) + 1; n_in_pair[y] = n_in_pair.get(y, 0) + 1
    for k in np.nonzero(has)[0]:
        j = idx[int(pg[k])]
        assert ((pos[k] - pos[j]) ** 2).sum() <= 2500
        assert a["species"][k] != a["species"][j]
        assert (min(int(a["id"][k]), int(pg[k])), max(int(a["id"][k]), int(pg[k]))) in pairs
    # pair draw is symmetric: for isolated pairs (each member in exactly one in-range pair)
    # proposals are mutual or absent together, and present with probability p_bind
    iso = [(x, y) for x, y in pairs if n_in_pair[x] == 1 and n_in_pair[y] == 1]
    assert len(iso) > 100
    both = 0
    for x, y in iso:
        px, py = pg[idx[x]], pg[idx[y]]
        assert (px == y) == (py == x)
        both += int(px == y)
    p = both / len(iso)
    assert abs(p - 0.5) < 4.5 * np.sqrt(0.25 / len(iso))


def test_bind_step_is_a_matching_with_anchor_rule():
    m = tiny_cube(L=300, n_a=1200, n_b=1200, cell=64, p_bind=0.9, p_rel=0.0)
    o = Oracle(m); o.seed_population(); o.debug_move_only()
    a = o.read_agents()
    prop = o.debug_proposals(MODE_BRUTE)
    idx = {int(i): k for k, i in enumerate(a["id"])}
    mutual = {(int(a["id"][k]), int(prop[k])) for k in range(len(prop))
              if prop[k] != NOPROP and prop[idx[int(prop[k])]] == a["id"][k]}
    anchors = {i for i, j in mutual if a["species"][idx[i]] == 0}
    dead = {i for i, j in mutual if a["species"][idx[i]] == 1}
    assert len(anchors) == len(dead) == len(mutual) // 2 > 20
    o2 = Oracle(m); o2.seed_population(); o2.step(1)
    b = o2.read_agents()
    ids_after = set(int(i) for i in b["id"])
    assert ids_after == set(range(2400)) - dead                                # S10: non-anchor dies
    assert {int(i) for i, s in zip(b["id"], b["species"]) if s == 2} == anchors  # anchor (A) becomes C
    ka = np.array([idx[i] for i in sorted(anchors)])
    kb = np.searchsorted(b["id"], sorted(anchors))
    for k in "xyz":
        assert (a[k][ka] == b[k][kb]).all()                                    # complex sits at the anchor


def test_results_independent_of_cell_size_and_memory_order():
    m = tiny_cube(L=400, n_a=1500, n_b=1500, p_rel=0.02)
    ref = None
    for cell, mode in [(50, MODE_GRID), (64, MODE_GRID), (400, MODE_GRID), (64, MODE_BRUTE)]:
        o = Oracle(m, cell_size=cell, mode=mode); o.seed_population(); o.step(12)
        s = (o.read_agents(), o.read_counts())
        if ref is None:
            ref = s
        assert state_equal(ref[0], s[0]) and (ref[1] == s[1]).all()
    # shuffled memory order (H1): every decision is keyed by id
    o = Oracle(m); o.seed_population(); a = o.read_agents()
    perm = np.random.default_rng(3).permutation(len(a["id"]))
    o2 = Oracle(m); o2.load_agents(*(a[k][perm] for k in ("x", "y", "z", "species", "id")))
    o2.step(12)
    assert state_equal(ref[0], o2.read_agents())


# --------------------------------------------------------------------------- unimolecular / births (S11,S13,S14)
def test_release_rate_is_binomial_and_ids_in_parent_order():
    m = tiny_cube(L=4000, n_a=1, n_b=1, p_bind=0.0, p_rel=0.01, cell=64)
    n = 100_000
    m.capacity = 2 * n; m.id_capacity = 3 * n
    rng = np.random.default_rng(5)
    pos = rng.integers(20, 3980, size=(3, n)).astype(np.int32)
    ids = rng.permutation(n).astype(np.uint32)            # memory order != id order
    o = Oracle(m)
    o.load_agents(pos[0], pos[1], pos[2], np.full(n, 2, np.uint16), ids, next_id=n)
    o.step(1)
    b = o.read_agents()
    n_new = len(b["id"]) - n
    assert abs(n_new - n * 0.01) < 4.5 * np.sqrt(n * 0.01 * 0.99)      # Bin(N, p)
    assert (b["id"] == np.arange(n + n_new)).all()                      # unique, contiguous newborn ids
    parents = np.nonzero(b["species"][:n] == 0)[0]                      # C -> A, keeps id (S11)
    assert len(parents) == n_new and (b["species"][n:] == 1).all()      # newborn = B
    for k in "xyz":                                                     # g-th newborn belongs to g-th parent by id (S14)
        d = b[k][n:].astype(np.int64) - b[k][parents].astype(np.int64)
        assert np.abs(d).max() <= 10 and d.min() < -5 and d.max() > 5   # +-1 nm offsets (S11)
    c = o.read_counts()[1, 0]
    assert list(c) == [n_new, n_new, n - n_new]


def test_degrade_and_channel_priority():
    # species X: ch0 = DEGRADE p=.3, ch1 = RELEASE p=1 -> release only when degrade did not fire (S13)
    X, Y, Z = 0, 1, 2
    sp = [Species("X", 0, channels=[Channel(CH_DEGRADE, prob_to_thr(0.3)), Channel(CH_RELEASE, prob_to_thr(1.0), Y, Z)]),
          Species("Y", 0), Species("Z", 0)]
    m = Model(name="prio", species=sp, reactions=[], compartments=[Compartment(SHAPE_CUBE, L=1000)],
              table_bits=12, tables=stack_tables([], 12), extent=(1000,) * 3, seed=77, place_seed=77,
              seed_records=[SeedRecord(X, 20000)], n_steps=4, cell_size=64).finalize()
    o = Oracle(m); o.seed_population(); o.step(1)
    c = o.read_counts()[1, 0]
    assert c[0] == 0 and c[1] == c[2]
    assert abs((20000 - c[1]) - 6000) < 4.5 * np.sqrt(20000 * 0.3 * 0.7)


def test_mean_complex_lifetime():
    m = tiny_cube(L=4000, n_a=1, n_b=1, p_bind=0.0, p_rel=0.02, cell=64)
    n = 20000
    m.capacity = 3 * n; m.id_capacity = 3 * n; m.counts_rows = 400
    pos = np.random.default_rng(8).integers(0, 4000, size=(3, n)).astype(np.int32)
    o = Oracle(m); o.load_agents(pos[0], pos[1], pos[2], np.full(n, 2, np.uint16), np.arange(n, dtype=np.uint32))
    o.step(300)
    c = o.read_counts()[:, 0, 2].astype(np.float64)
    # survival (1-p)^t ; mean lifetime 1/p = 50 steps
    assert abs(c[50] / n - 0.98**50) < 0.015 and abs(c[150] / n - 0.98**150) < 0.01


# --------------------------------------------------------------------------- conservation (north_star)
def test_moiety_conservation_w0_every_step():
    m = configs.w0(cell_size=512, n_steps=300)
    o = Oracle(m); o.seed_population(); o.step(300)
    c = o.read_counts()[:, 0, :].astype(np.int64)
    assert (c[:, 0] + c[:, 2] == 5000).all() and (c[:, 1] + c[:, 2] == 5000).all()
    assert c[300, 2] > 500
    assert c.sum(axis=1)[-1] == o.info()["n_live"]


def cascade_totals(m, c):
    ix = {s.name: i for i, s in enumerate(m.species)}
    g = lambda *names: sum(c[..., ix[n]] for n in names if n in ix)
    return {
        "BRAF": g("BRAF", "BRAF:MEK", "BRAF:INH"),
        "MEK": g("MEK", "pMEK", "BRAF:MEK", "pMEK:ERK", "P:pMEK"),
        "ERK": g("ERK", "pERK", "pMEK:ERK", "P:pERK"),
        "P": g("P", "P:pMEK", "P:pERK"),
        "INH": g("INH", "BRAF:INH"),
    }


def test_moiety_conservation_cascade_with_replicas():
    m = configs.w2(scale=0.002, n_steps=150)      # 8 replicas, ~17.7 k agents, dense enough to react
    # shrink the spheres further so that reactions happen within 150 steps
    o = Oracle(m); o.seed_population(); o.step(150)
    c = o.read_counts().astype(np.int64)          # [row][replica][species]
    tot = cascade_totals(m, c)
    for k, v in tot.items():
        assert (v == v[0]).all(), k               # constant in time, per replica
    assert tot["INH"][0, 0] == 0 and tot["INH"][0, 7] == 630
    ix = {s.name: i for i, s in enumerate(m.species)}
    assert c[-1, :, ix["BRAF:MEK"]].sum() + c[-1, :, ix["pMEK"]].sum() > 0
    assert c[-1].sum() == o.info()["n_live"]
    a = o.read_agents()
    assert ((a["x"] >> m.stride_shift) < 8).all()


# --------------------------------------------------------------------------- checkpoint
def test_step_a_then_b_equals_step_a_plus_b():
    m = tiny_cube(L=400, n_a=1500, n_b=1500, p_rel=0.02)
    o = Oracle(m); o.seed_population(); o.step(5); o.step(9)
    o2 = Oracle(m); o2.seed_population(); o2.step(14)
    assert state_equal(o.read_agents(), o2.read_agents()) and (o.read_counts() == o2.read_counts()).all()
    # dump / reload
    o3 = Oracle(m); o3.seed_population(); o3.step(5)
    a = o3.read_agents(); inf = o3.info()
    o4 = Oracle(m); o4.load_agents(a["x"], a["y"], a["z"], a["species"], a["id"], step=5, next_id=inf["next_id"])
    o4.step(9)
    assert state_equal(o4.read_agents(), o2.read_agents())


# --------------------------------------------------------------------------- W3 structure (S7,S17)
def test_w3_expression_delay_and_blocking():
    m = configs.w3(scale=0.004, n_steps=900, delay=40, cell_size=256)
    ix = {s.name: i for i, s in enumerate(m.species)}
    # make the nuclear events frequent enough for a short test: start with pERK_n next to the genes
    o = Oracle(m); o.seed_population()
    a = o.read_agents()
    genes = np.nonzero(a["species"] == ix["GENE"])[0]
    assert len(genes) == 2
    extra = 400
    n0 = len(a["id"])
    rng = np.random.default_rng(1)
    ex = {k: np.concatenate([a[k], (a[k][genes[rng.integers(0, 2, extra)]] + rng.integers(-60, 60, extra)).astype(np.int32)])
          for k in "xyz"}
    sp = np.concatenate([a["species"], np.full(extra, ix["pERK_n"], np.uint16)])
    ids = np.concatenate([a["id"], np.arange(n0, n0 + extra, dtype=np.uint32)])
    o.load_agents(ex["x"], ex["y"], ex["z"], sp, ids)
    gene_pos = {k: a[k][genes].copy() for k in "xyz"}
    o.step(900)
    c = o.read_counts()[:, 0, :].astype(np.int64)
    tf = o.info()["t_first0"]
    assert tf != 0xFFFFFFFF
    made = c[:, ix["mRNA_n"]] + c[:, ix["mRNA_c"]]
    assert (made[: tf + 1] == 0).all() and made[tf + 1] >= 1                 # first transcription at step tf
    F_tot = c[:, ix["F_n"]] + c[:, ix["GENE:F"]]
    assert (F_tot[: tf + 40 + 1] == 0).all() and (F_tot[tf + 40 + 1:] == 2).all()  # S17: one F per locus at tf+delay
    locus = c[:, ix["GENE"]] + c[:, ix["GENE:pERK"]] + c[:, ix["GENE:F"]]
    assert (locus == 2).all()
    b = o.read_agents()
    gl = np.isin(b["species"], [ix["GENE"], ix["GENE:pERK"], ix["GENE:F"]])
    for k in "xyz":
        assert sorted(b[k][gl]) == sorted(gene_pos[k])                        # loci never move (S10)
    # compartment invariant for every agent
    R = m.compartments[0].r_out; Rn = m.compartments[1].r_out
    r2 = sum((b[k].astype(np.int64) - R) ** 2 for k in "xyz")
    comp = np.array([s.compartment for s in m.species])[b["species"]]
    assert ((r2[comp == 0] > Rn * Rn) & (r2[comp == 0] <= R * R)).all() and (r2[comp == 1] <= Rn * Rn).all()


# --------------------------------------------------------------------------- validation
def test_create_validation():
    def bad(mut):
        m = tiny_cube()
        mut(m)
        with pytest.raises(OracleError) as e:
            Oracle(m)
        assert e.value.code == E_INVAL

    bad(lambda m: m.reactions.append(Reaction(1, 0, 2, 2500, 1)))           # duplicate unordered pair
    bad(lambda m: setattr(m.reactions[0], "cplx", 9))                       # missing species
    bad(lambda m: setattr(m, "cell_size", 49))                              # cell smaller than R
    bad(lambda m: setattr(m.species[2].channels[0], "prod1", 7))            # product does not exist
    bad(lambda m: setattr(m.compartments[0], "L", 100))                     # table reaches past the domain
    Oracle(tiny_cube())


# --------------------------------------------------------------------------- equilibrium (north_star)
@pytest.mark.slow
def test_w0_mass_action_equilibrium():
    """Long-run C near the mass-action equilibrium: (5000-C)^2 = (k_b/k_f) C with
    k_f = p_bind (4/3) pi R^3 / V = 2.618e-7, k_b = 1e-3  ->  C_eq = 2140.6."""
    kf = 0.5 * 4.0 / 3.0 * np.pi * 5.0**3 / 1e9
    K = 1e-3 / kf
    c_eq = ((2 * 5000 + K) - np.sqrt((2 * 5000 + K) ** 2 - 4 * 5000**2)) / 2
    assert abs(c_eq - 2140.6) < 0.5
    m = configs.w0(cell_size=512, n_steps=8000)
    o = Oracle(m); o.seed_population(); o.step(8000)
    c = o.read_counts()[:, 0, 2].astype(np.float64)
    mean_c = c[4000:].mean()
    assert 2080 <= mean_c <= 2200, mean_c
    assert 1850 <= c[1000] <= 2000        # the 1,000 steps of [CFG 0] are still relaxing
