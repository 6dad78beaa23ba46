"""Full-length runs of the BASELINE.json workloads on the CUDA path, checked by properties that hold at any
size (the oracle cannot follow these lengths in test time): moiety conservation on EVERY counts row, the
compartment invariant, id bookkeeping, and for [CFG 0] the mass-action equilibrium of north_star.
The same properties pin the oracle on CPU (tests/test_oracle_pins.py); bit-exact agreement of the two on
shorter runs is in tests/test_gpu_parity.py."""
import numpy as np
import pytest

from workloads import configs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_14603_b200 as pkg

    pkg.load_library()
    return pkg


def cascade_totals(m, c):
    ix = {s.name: i for i, s in enumerate(m.species)}
    g = lambda *names: sum(c[..., ix[n]] for n in names if n in ix)
    return {"BRAF": g("BRAF", "BRAF:MEK", "BRAF:INH"),
            "MEK": g("MEK", "pMEK", "BRAF:MEK", "pMEK:ERK", "P:pMEK"),
            "ERK": g("ERK", "pERK", "pMEK:ERK", "P:pERK"),
            "P": g("P", "P:pMEK", "P:pERK"),
            "INH": g("INH", "BRAF:INH")}


def check_ids_and_positions(sim, m):
    a, info = sim.read_agents(), sim.info()
    assert len(a["id"]) == info["n_live"]
    assert (np.diff(a["id"].astype(np.int64)) > 0).all() and a["id"][-1] < info["next_id"]
    for k, ext in zip("xyz", m.extent):
        assert a[k].min() >= 0 and a[k].max() < ext
    return a


def test_w0_full_length_equilibrium(gpu):
    """[CFG 0] for 12,000 steps: A+C and B+C constant on every row; mean C over the second half inside the
    band around the mass-action equilibrium C_eq = 2140.6 (same band as the oracle pin)."""
    m = configs.w0(cell_size=448, n_steps=12000)
    sim = gpu.Sim(m); sim.seed_population(); sim.step(12000)
    c = sim.read_counts()[:, 0, :].astype(np.int64)
    assert c.shape[0] == 12001
    assert (c[:, 0] + c[:, 2] == 5000).all() and (c[:, 1] + c[:, 2] == 5000).all()
    mean_c = c[6000:, 2].mean()
    assert 2080 <= mean_c <= 2200, mean_c
    assert 1850 <= c[1000, 2] <= 2000
    check_ids_and_positions(sim, m)


def test_w1_full_size_full_length_conservation(gpu):
    """[CFG 1] in full: 1.05 M agents, 10,000 steps, per-step counts recorded."""
    m = configs.w1()
    sim = gpu.Sim(m); sim.seed_population(); sim.step(10000)
    c = sim.read_counts().astype(np.int64)
    assert c.shape[0] == 10001
    for k, v in cascade_totals(m, c).items():
        if np.ndim(v) == 0:
            continue                      # moiety not in this model
        assert (v == v[0]).all(), k
    ix = {s.name: i for i, s in enumerate(m.species)}
    assert c[-1, 0, ix["pERK"]] > 0 and c[-1, 0, ix["pMEK"]] > 0          # the cascade fired
    a = check_ids_and_positions(sim, m)
    cmp = m.compartments[0]
    r2 = (a["x"].astype(np.int64) - cmp.cx) ** 2 + (a["y"].astype(np.int64) - cmp.cy) ** 2 + \
         (a["z"].astype(np.int64) - cmp.cz) ** 2
    assert (r2 <= cmp.r_out ** 2).all()                                    # nobody left the sphere


@pytest.mark.slow
def test_w2_full_size_dose_sweep(gpu):
    """[CFG 2] in full: 8 replicas, 8.85 M agents, 5,000 steps; totals conserved per replica on every row,
    agents never leave their replica tile, and the steady-state pERK fraction falls with the dose."""
    m = configs.w2()
    sim = gpu.Sim(m); sim.seed_population(); sim.step(5000)
    c = sim.read_counts().astype(np.int64)
    for k, v in cascade_totals(m, c).items():
        if np.ndim(v) == 0:
            continue                      # moiety not in this model
        assert (v == v[0]).all(), k
    ix = {s.name: i for i, s in enumerate(m.species)}
    frac = c[-500:, :, ix["pERK"]].mean(axis=0) / 600000.0                 # reading S19
    assert frac[0] > 0 and frac[7] < frac[0]
    a = sim.read_agents()
    assert ((a["x"] >> m.stride_shift) < 8).all()


def test_w3_full_size_expression(gpu):
    """[CFG 3] at full size for 6,000 steps (with the 50 nm gene locus and primed nuclear pERK of the trace recipe, so
    that transcription starts: workloads/configs.py w3): compartment invariant for every agent, mRNA appears, exported
    and translated, and the delayed repressor is born exactly `delay` = 2,000 steps after the first transcription,
    one per gene locus.  Nothing here is conditional."""
    delay = 2000
    m = configs.w3(n_steps=6000, delay=delay, gene_radius=500, primed_perk_n=2000)
    sim = gpu.Sim(m); sim.seed_population(); sim.step(6000)
    c = sim.read_counts()[:, 0, :].astype(np.int64)
    ix = {s.name: i for i, s in enumerate(m.species)}
    a = check_ids_and_positions(sim, m)
    comp_of = np.array([s.compartment for s in m.species])
    for k, cmp in enumerate(m.compartments):
        sel = comp_of[a["species"]] == k
        r2 = (a["x"][sel].astype(np.int64) - cmp.cx) ** 2 + (a["y"][sel].astype(np.int64) - cmp.cy) ** 2 + \
             (a["z"][sel].astype(np.int64) - cmp.cz) ** 2
        assert (r2 <= cmp.r_out ** 2).all()
        if cmp.r_in >= 0:
            assert (r2 > cmp.r_in ** 2).all()
    assert (c[:, ix["GENE"]] + c[:, ix["GENE:pERK"]] + c[:, ix["GENE:F"]] == 2).all()      # the two fixed loci
    t_first = sim.info()["t_first0"]
    assert t_first != 0xFFFFFFFF and t_first + delay + 1 < 6000, t_first
    assert c[:t_first + 1, ix["mRNA_n"]].max() == 0 and c[t_first + 1, ix["mRNA_n"]] >= 1   # first transcription at t_first
    assert c[:, ix["mRNA_c"]].max() > 0 and c[:, ix["cFos_c"]].max() > 0                    # export and translation
    rep = c[:, ix["F_n"]] + c[:, ix["GENE:F"]]
    assert (rep[:t_first + delay + 1] == 0).all() and (rep[t_first + delay + 1:] == 2).all()  # born at t_first + delay


@pytest.mark.parametrize("n", [1_000_000, 4_000_000, 16_000_000, pytest.param(64_000_000, marks=pytest.mark.slow)])
def test_w4_all_sizes_100_steps(gpu, n):
    """[CFG 4]: every N for its 100 steps; A+C and B+C constant on every row, live agents = row sum, and the
    complex density after 100 steps inside the band of the float Monte-Carlo estimate (~3,700 per um^3)."""
    m = configs.w4(n=n, n_steps=100)
    sim = gpu.Sim(m); sim.seed_population(); sim.step(100)
    c = sim.read_counts()[:, 0, :].astype(np.int64)
    assert c.shape[0] == 101
    assert (c[:, 0] + c[:, 2] == n // 2).all() and (c[:, 1] + c[:, 2] == n // 2).all()
    assert c[-1].sum() == sim.info()["n_live"]
    density = c[-1, 2] / (n / 30000.0)
    assert 3300 <= density <= 4100, density
    assert (np.diff(c[:, 2]) > 0).all()          # far from equilibrium: C grows every step at these sizes
