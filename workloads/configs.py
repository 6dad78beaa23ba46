"""The five synthetic workloads of BASELINE.json `configs` (W0..W4), as integer Models.

All inputs are seeded and synthetic; they stand in for the paper's dabrafenib /
MAPK run (section 3.1, Table 1) and its cFos run (PAPER.md:153-167,
section 3.4), whose reaction sets and rate constants are not in PAPER.md.
Parameter choices where BASELINE.json leaves a range are reading S18 of DESIGN.md.
"""
from __future__ import annotations

from .model import (CH_BIRTH, CH_DEGRADE, CH_DELAYED_BIRTH, CH_RELEASE, NONE16,
                    SHAPE_CUBE, SHAPE_SPHERE, Channel, Compartment, Model,
                    Reaction, SeedRecord, Species, prob_to_thr, sigma_units,
                    stack_tables)

TABLE_BITS = 12
R_BIND = 50                # 5 nm in 0.1 nm units
R2_BIND = R_BIND * R_BIND  # 2,500


def _release(p, prod0, prod1):
    return Channel(CH_RELEASE, prob_to_thr(p), prod0, prod1)


# ----------------------------------------------------------------------------- W0 / W4
def ab_c_cube(L: int, n_a: int, n_b: int, *, seed: int, place_seed: int, n_steps: int,
              cell_size: int, name: str) -> Model:
    """A + B <-> C in a reflective cube [CFG 0, CFG 4]."""
    A, B, C = 0, 1, 2
    sig_free = sigma_units(10.0, 1.0)   # 44.72 units
    sig_c = sigma_units(5.0, 1.0)       # 31.62 units
    species = [
        Species("A", sigma_class=1),
        Species("B", sigma_class=1),
        Species("C", sigma_class=2, channels=[_release(1e-3, A, B)]),
    ]
    m = Model(
        name=name, species=species,
        reactions=[Reaction(A, B, C, R2_BIND, prob_to_thr(0.5))],
        compartments=[Compartment(SHAPE_CUBE, L=L)],
        table_bits=TABLE_BITS, tables=stack_tables([sig_free, sig_c], TABLE_BITS),
        extent=(L, L, L), seed=seed, place_seed=place_seed,
        seed_records=[SeedRecord(A, n_a), SeedRecord(B, n_b)],
        n_steps=n_steps, cell_size=cell_size, dt_us=1.0,
        volume_um3=(L / 10_000.0) ** 3,
    )
    return m.finalize()


def w0(cell_size: int = 50, n_steps: int = 1000, seed: int = 1) -> Model:
    """[CFG 0]: 5,000 A + 5,000 B, 1 um cube, 5 nm cells as stated in the config."""
    return ab_c_cube(10_000, 5_000, 5_000, seed=seed, place_seed=seed, n_steps=n_steps,
                     cell_size=cell_size, name="W0_toy_AB_C")


W4_EDGES = {1_000_000: 32_183, 4_000_000: 51_087, 16_000_000: 81_096, 64_000_000: 128_732}


def w4(n: int = 16_000_000, cell_size: int = 448, n_steps: int = 100) -> Model:
    """[CFG 4]: fixed density 30,000 agents/um^3 (reading S21 for the cube edges)."""
    if n in W4_EDGES:
        L = W4_EDGES[n]
    else:  # other sizes (tests): same density, edge rounded to the lattice
        L = int(round((n / 30_000.0) ** (1.0 / 3.0) * 10_000))
    return ab_c_cube(L, n // 2, n - n // 2, seed=5, place_seed=5, n_steps=n_steps,
                     cell_size=cell_size, name=f"W4_scaling_{n}")


# ----------------------------------------------------------------------------- W1 / W2
def _cascade_species(sig_free_cls=1, sig_cplx_cls=2, comp=0, rel_p=2e-3):
    """BRAF -> MEK -> ERK cascade with one phosphatase [CFG 1]. Returns (species, reactions)."""
    names = ["BRAF", "MEK", "ERK", "P", "pMEK", "pERK",
             "BRAF:MEK", "pMEK:ERK", "P:pMEK", "P:pERK"]
    ix = {n: i for i, n in enumerate(names)}
    sp = [Species(n, sigma_class=sig_free_cls, compartment=comp) for n in names[:6]]
    sp += [
        Species("BRAF:MEK", sig_cplx_cls, comp, channels=[_release(rel_p, ix["BRAF"], ix["pMEK"])]),
        Species("pMEK:ERK", sig_cplx_cls, comp, channels=[_release(rel_p, ix["pMEK"], ix["pERK"])]),
        Species("P:pMEK", sig_cplx_cls, comp, channels=[_release(rel_p, ix["P"], ix["MEK"])]),
        Species("P:pERK", sig_cplx_cls, comp, channels=[_release(rel_p, ix["P"], ix["ERK"])]),
    ]
    rx = [
        Reaction(ix["BRAF"], ix["MEK"], ix["BRAF:MEK"], R2_BIND, prob_to_thr(0.8)),
        Reaction(ix["pMEK"], ix["ERK"], ix["pMEK:ERK"], R2_BIND, prob_to_thr(0.6)),
        Reaction(ix["P"], ix["pMEK"], ix["P:pMEK"], R2_BIND, prob_to_thr(0.3)),
        Reaction(ix["P"], ix["pERK"], ix["P:pERK"], R2_BIND, prob_to_thr(0.3)),
    ]
    return sp, rx, ix


SPHERE_R = 50_000  # 5 um


def w1(scale: float = 1.0, n_steps: int = 10_000, cell_size: int = 1024, seed: int = 2) -> Model:
    """[CFG 1]: MAPK/ERK-shaped cascade in one reflective sphere, ~1.05 M agents.

    `scale` < 1 shrinks counts and volume together (fixed concentration; the
    paper's volume down-scaling) for tests.
    """
    sp, rx, ix = _cascade_species()
    R = int(round(SPHERE_R * scale ** (1.0 / 3.0)))
    counts = [("BRAF", 50_000), ("MEK", 300_000), ("ERK", 600_000), ("P", 100_000)]
    recs = [SeedRecord(ix[n], max(1, int(round(c * scale)))) for n, c in counts]
    m = Model(
        name="W1_mapk_sphere", species=sp, reactions=rx,
        compartments=[Compartment(SHAPE_SPHERE, R, R, R, r_out=R)],
        table_bits=TABLE_BITS,
        tables=stack_tables([sigma_units(4.0, 10.0), sigma_units(2.0, 10.0)], TABLE_BITS),
        extent=(2 * R + 1,) * 3, seed=seed, place_seed=seed, seed_records=recs,
        n_steps=n_steps, cell_size=cell_size, dt_us=10.0,
        volume_um3=4.0 / 3.0 * 3.141592653589793 * (R / 10_000.0) ** 3,
    )
    return m.finalize()


W2_INHIBITOR = [0, 315, 945, 3_150, 9_450, 31_500, 94_500, 315_000]


def w2(scale: float = 1.0, n_steps: int = 5_000, cell_size: int = 1024, seed: int = 3) -> Model:
    """[CFG 2]: eight dose replicas tiled along x (reading S16), ~8.85 M agents."""
    sp, rx, ix = _cascade_species()
    INH, BRAF_INH = len(sp), len(sp) + 1
    sp.append(Species("INH", sigma_class=3))
    sp.append(Species("BRAF:INH", sigma_class=2, channels=[_release(1e-4, ix["BRAF"], INH)]))
    rx.append(Reaction(ix["BRAF"], INH, BRAF_INH, R2_BIND, prob_to_thr(0.9)))
    R = int(round(SPHERE_R * scale ** (1.0 / 3.0)))
    stride_shift = 17
    assert 2 * R + 1 + 4 * R_BIND < (1 << stride_shift)
    counts = [("BRAF", 50_000), ("MEK", 300_000), ("ERK", 600_000), ("P", 100_000)]
    recs = []
    for rep, n_inh in enumerate(W2_INHIBITOR):
        recs += [SeedRecord(ix[n], max(1, int(round(c * scale))), rep) for n, c in counts]
        k = int(round(n_inh * scale))
        if k:
            recs.append(SeedRecord(INH, k, rep))
    m = Model(
        name="W2_dose_sweep", species=sp, reactions=rx,
        compartments=[Compartment(SHAPE_SPHERE, R, R, R, r_out=R)],
        table_bits=TABLE_BITS,
        tables=stack_tables([sigma_units(4.0, 1.0), sigma_units(2.0, 1.0),
                             sigma_units(50.0, 1.0)], TABLE_BITS),
        extent=(8 << stride_shift, 2 * R + 1, 2 * R + 1), seed=seed, place_seed=seed,
        seed_records=recs, n_steps=n_steps, cell_size=cell_size,
        n_replicas=8, stride_shift=stride_shift, dt_us=1.0,
        volume_um3=4.0 / 3.0 * 3.141592653589793 * (R / 10_000.0) ** 3,
    )
    return m.finalize()


# ----------------------------------------------------------------------------- W3
def w3(scale: float = 1.0, n_steps: int = 20_000, cell_size: int = 1024, seed: int = 4,
       delay: int = 2_000, gene_radius: int = R_BIND, primed_perk_n: int = 0) -> Model:
    """[CFG 3]: cytoplasm shell + nucleus, membrane crossing, expression, delayed repressor.

    `gene_radius` (units) is the capture radius of the two gene-locus agents for nuclear pERK and for the repressor.
    [CFG 3] gives none; reading S18 takes the 5 nm of the other reactions, with which a full-size run practically never
    transcribes (a few dozen nuclear pERK against two 5 nm targets in 65 um^3).  The long-run parity trace
    (tests/golden/make_traces.py) therefore uses a 50 nm locus, `primed_perk_n` nuclear pERK seeded at t = 0 and a
    200-step delay, so that the expression branch and the delayed rule run at full size inside a trace the oracle can
    produce; parity does not depend on the values."""
    CYT, NUC = 0, 1
    sp, rx, ix = _cascade_species(comp=CYT)

    def add(s: Species) -> int:
        sp.append(s)
        ix[s.name] = len(sp) - 1
        return len(sp) - 1

    p_rel = 2e-3
    pERK_c = ix["pERK"]
    RSK = add(Species("RSK", 1, CYT))
    pRSK_c = add(Species("pRSK_c", 1, CYT))
    pERK_n = add(Species("pERK_n", 1, NUC))
    pRSK_n = add(Species("pRSK_n", 1, NUC))
    # membrane crossing (reading S7): bidirectional with the same p per contact
    thr_x = prob_to_thr(0.05)
    sp[pERK_c].cross_to, sp[pERK_c].cross_thr = pERK_n, thr_x
    sp[pERK_n].cross_to, sp[pERK_n].cross_thr = pERK_c, thr_x
    sp[pRSK_c].cross_to, sp[pRSK_c].cross_thr = pRSK_n, thr_x
    sp[pRSK_n].cross_to, sp[pRSK_n].cross_thr = pRSK_c, thr_x
    pERK_RSK = add(Species("pERK:RSK", 2, CYT, channels=[_release(p_rel, pERK_c, pRSK_c)]))
    rx.append(Reaction(pERK_c, RSK, pERK_RSK, R2_BIND, prob_to_thr(0.5)))

    mRNA_c = add(Species("mRNA_c", 1, CYT))
    mRNA_n = add(Species("mRNA_n", 1, NUC, cross_to=mRNA_c, cross_thr=prob_to_thr(0.02),
                         channels=[Channel(CH_DEGRADE, prob_to_thr(5e-5))]))
    cFos = add(Species("cFos_c", 1, CYT, channels=[Channel(CH_DEGRADE, prob_to_thr(2e-5))]))
    pcFos = add(Species("pcFos_c", 1, CYT, channels=[Channel(CH_DEGRADE, prob_to_thr(2e-5))]))
    sp[mRNA_c].channels = [Channel(CH_BIRTH, prob_to_thr(1e-3), prod1=cFos),
                           Channel(CH_DEGRADE, prob_to_thr(5e-5))]
    pERK_cFos = add(Species("pERK:cFos", 2, CYT, channels=[_release(p_rel, pERK_c, pcFos)]))
    rx.append(Reaction(pERK_c, cFos, pERK_cFos, R2_BIND, prob_to_thr(0.5)))

    F_n = add(Species("F_n", 1, NUC))
    GENE = add(Species("GENE", 0, NUC))
    GENE_pERK = add(Species("GENE:pERK", 0, NUC))
    GENE_F = add(Species("GENE:F", 0, NUC))   # permanently blocked locus (reading S17)
    emit_F = Channel(CH_DELAYED_BIRTH, delay, prod1=F_n, rule=0)
    sp[GENE].channels = [emit_F]
    sp[GENE_pERK].channels = [
        Channel(CH_BIRTH, prob_to_thr(0.01), prod1=mRNA_n, rule=0, marks_first=True),
        _release(p_rel, GENE, pERK_n),
        emit_F,
    ]
    rx.append(Reaction(GENE, pERK_n, GENE_pERK, gene_radius * gene_radius, prob_to_thr(0.5)))
    rx.append(Reaction(GENE, F_n, GENE_F, gene_radius * gene_radius, prob_to_thr(0.5)))

    R = int(round(SPHERE_R * scale ** (1.0 / 3.0)))
    Rn = R // 2
    counts = [("BRAF", 12_500), ("MEK", 75_000), ("ERK", 150_000), ("P", 25_000), ("RSK", 75_000)]
    recs = [SeedRecord(ix[n], max(1, int(round(c * scale)))) for n, c in counts]
    recs.append(SeedRecord(GENE, 2))
    if primed_perk_n:
        recs.append(SeedRecord(pERK_n, primed_perk_n))
    m = Model(
        name="W3_nuclear", species=sp, reactions=rx,
        compartments=[Compartment(SHAPE_SPHERE, R, R, R, r_out=R, r_in=Rn),
                      Compartment(SHAPE_SPHERE, R, R, R, r_out=Rn)],
        table_bits=TABLE_BITS,
        tables=stack_tables([sigma_units(4.0, 10.0), sigma_units(2.0, 10.0)], TABLE_BITS),
        extent=(2 * R + 1,) * 3, seed=seed, place_seed=seed, seed_records=recs,
        n_steps=n_steps, cell_size=cell_size, n_rules=1, dt_us=10.0,
        volume_um3=4.0 / 3.0 * 3.141592653589793 * (R / 10_000.0) ** 3,
    )
    m.capacity = int(m.n_agents0 * 1.6) + 4096
    m.id_capacity = int(m.n_agents0 * 4) + 65536
    return m.finalize()


def by_name(name: str, **kw) -> Model:
    return {"w0": w0, "w1": w1, "w2": w2, "w3": w3, "w4": w4}[name.lower()](**kw)
