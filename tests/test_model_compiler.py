"""Model compiler from physical units (workloads/compiler.py).  CPU only."""
import json
import math

import numpy as np
import pytest

from workloads import compiler, model


def toy(**kw):
    spec = {
        "name": "toy", "volume_l": 1e-15, "dt_us": 1.0, "seed": 7, "n_steps": 50,     # 1 fL = 1 um^3
        "molecules": [
            {"name": "A", "mw_da": 40_000, "concentration_molar": 8.3e-6,
             "interactions": [{"partner": "B", "complex": "C", "radius_nm": 5.0, "p_bind": 0.5}]},
            {"name": "B", "mw_da": 40_000, "concentration_molar": 8.3e-6,
             "interactions": [{"partner": "A", "complex": "C", "radius_nm": 5.0, "p_bind": 0.5}]},
            {"name": "C", "mw_da": 80_000, "release": {"kcat_per_s": 1000.0, "products": ["A", "B"]}},
        ],
    }
    spec.update(kw)
    return spec


def test_closed_forms():
    # Stokes-Einstein: a 1 nm sphere in water at 25 C (eta = 0.89 mPa s): D = kT / (6 pi eta r) = 2.45e-10 m^2/s
    d = compiler.stokes_einstein_um2_s(1.0, 298.15, 8.9e-4)
    assert abs(d - 245.4) < 0.5
    assert abs(compiler.stokes_einstein_um2_s(2.0, 298.15, 8.9e-4) - d / 2) < 1e-9          # D ~ 1 / r
    # radius ~ MW^(1/3): 8x the weight, 2x the radius; a 50 kDa protein is about 2.4 nm
    assert abs(compiler.radius_nm(8 * 50_000) / compiler.radius_nm(50_000) - 2.0) < 1e-12
    assert abs(compiler.radius_nm(50_000) - 2.43) < 0.01
    # turnover: p = 1 - exp(-k dt) -> k dt for small k dt, 1 for large
    assert abs(compiler.kcat_to_prob(1000.0, 1.0) - (1 - math.exp(-1e-3))) < 1e-15
    assert abs(compiler.kcat_to_prob(2.0, 10.0) / 2e-5 - 1.0) < 1e-4
    assert compiler.kcat_to_prob(1e12, 1.0) == 1.0
    # count = c N_A V (Table 1 in 3e-12 L)
    assert compiler.count_from_concentration(3e-9, 3e-12) == 5420
    assert compiler.count_from_concentration(1.2e-6, 3e-12) == 2167971


def test_compiled_tables():
    m = compiler.compile_model(json.dumps(toy()))
    assert m.extent == (10_000, 10_000, 10_000)                  # 1 um^3 -> 1 um edge = 10,000 units
    n = compiler.count_from_concentration(8.3e-6, 1e-15)
    assert [r.count for r in m.seed_records] == [n, n] and n == 4998
    # A and B share a sigma class, the heavier complex gets its own, narrower one
    assert m.species[0].sigma_class == m.species[1].sigma_class != m.species[2].sigma_class
    d_a = compiler.stokes_einstein_um2_s(compiler.radius_nm(40_000))
    var = (m.tables[m.species[0].sigma_class].astype(np.float64) ** 2).mean()
    assert abs(var / model.sigma_units(d_a, 1.0) ** 2 - 1.0) < 2e-3        # table variance = 2 D dt
    assert m.tables[m.species[2].sigma_class].max() < m.tables[m.species[0].sigma_class].max()
    (rx,) = m.reactions
    assert (rx.a, rx.b, rx.cplx, rx.r2, rx.thr) == (0, 1, 2, 2500, model.prob_to_thr(0.5))
    (ch,) = m.species[2].channels
    assert (ch.kind, ch.prod0, ch.prod1) == (model.CH_RELEASE, 0, 1)
    assert ch.thr == model.prob_to_thr(1 - math.exp(-1e-3))


def test_consistency_checker_findings():
    assert compiler.check(toy()) == []
    s = toy(); s["molecules"][1]["interactions"] = []
    assert any("no reciprocal" in f for f in compiler.check(s))
    s = toy(); s["molecules"][0]["interactions"][0]["complex"] = "Z"
    assert any("unknown molecule 'Z'" in f for f in compiler.check(s))
    s = toy(); s["molecules"][2]["mw_da"] = 3.0
    assert any("not plausible" in f for f in compiler.check(s))
    s = toy(volume_l=1e-21)
    assert any("less than one molecule" in f for f in compiler.check(s))
    s = toy(); s["molecules"][2]["release"]["products"] = ["A"]
    assert any("exactly two products" in f for f in compiler.check(s))
    with pytest.raises(compiler.ModelError):
        compiler.compile_model(s)


def test_compiled_model_runs_on_the_oracle_and_conserves_moieties():
    from oracle.binding import Oracle

    m = compiler.compile_model(toy(), cell_size=64)
    o = Oracle(m); o.seed_population(); o.step(50)
    c = o.read_counts()[:, 0, :].astype(np.int64)
    assert (c[:, 0] + c[:, 2] == c[0, 0]).all() and (c[:, 1] + c[:, 2] == c[0, 1]).all()
    assert c[-1, 2] > 0                                            # bindings happened


# --------------------------------------------------------------------------- localisation, translocation, expressors
def nuclear_spec(**over):
    """A [CFG 3]-shaped model in physical units: kinase K phosphorylates S in the cytosol,
    pS shuttles through the nuclear membrane, binds the gene locus, the bound locus expresses mRNA, which is
    exported, translated by an expressor reaction and degraded."""
    spec = {
        "name": "nuclear_physical", "dt_us": 10.0, "seed": 21, "n_steps": 40,
        "cell": {"radius_um": 0.6, "nucleus_radius_um": 0.3},
        "molecules": [
            {"name": "K", "mw_da": 85_000, "concentration_molar": 2.0e-6,
             "interactions": [{"partner": "S", "complex": "K:S", "radius_nm": 5.0, "p_bind": 0.8}]},
            {"name": "S", "mw_da": 42_000, "concentration_molar": 8.0e-6,
             "interactions": [{"partner": "K", "complex": "K:S", "radius_nm": 5.0, "p_bind": 0.8}]},
            {"name": "K:S", "mw_da": 127_000, "release": {"kcat_per_s": 5_000.0, "products": ["K", "pS"]}},
            {"name": "pS", "mw_da": 42_000, "translocation": {"to": "pS_n", "prob_per_contact": 0.05}},
            {"name": "pS_n", "mw_da": 42_000, "localisation": "nucleus", "concentration_molar": 3.0e-6,
             "translocation": {"to": "pS", "prob_per_contact": 0.05},
             "interactions": [{"partner": "GENE", "complex": "GENE:pS", "radius_nm": 40.0, "p_bind": 0.5}]},
            {"name": "GENE", "mw_da": 1_000_000, "localisation": "nucleus", "immobile": True, "count": 2,
             "interactions": [{"partner": "pS_n", "complex": "GENE:pS", "radius_nm": 40.0, "p_bind": 0.5}]},
            {"name": "GENE:pS", "mw_da": 1_042_000, "localisation": "nucleus", "immobile": True,
             "expression": {"product": "mRNA_n", "rate_per_s": 20_000.0},
             "release": {"kcat_per_s": 200.0, "products": ["GENE", "pS_n"]}},
            {"name": "mRNA_n", "mw_da": 400_000, "localisation": "nucleus", "degradation_per_s": 5.0,
             "translocation": {"to": "mRNA_c", "prob_per_contact": 0.02}},
            {"name": "mRNA_c", "mw_da": 400_000, "degradation_per_s": 5.0,
             "expression": {"product": "P", "rate_per_s": 100.0}},
            {"name": "P", "mw_da": 40_000, "degradation_per_s": 2.0},
        ],
    }
    spec.update(over)
    return spec


def test_compartmentalised_model_compiles_to_shell_nucleus_twins_and_channels():
    spec = nuclear_spec()
    assert compiler.check(spec) == []
    m = compiler.compile_model(spec, cell_size=512)
    R, Rn = 6000, 3000
    shell, nuc = m.compartments
    assert (shell.shape, shell.r_out, shell.r_in, nuc.r_out, nuc.r_in) == (model.SHAPE_SPHERE, R, Rn, Rn, -1)
    assert m.extent == (2 * R + 1,) * 3
    ix = {s.name: i for i, s in enumerate(m.species)}
    assert [m.species[ix[n]].compartment for n in ("K", "pS", "pS_n", "GENE", "mRNA_n", "mRNA_c")] == [0, 0, 1, 1, 1, 0]
    # counts: concentration x volume of the molecule's OWN compartment (closed form)
    v_cyt = 4.0 / 3.0 * math.pi * (0.6 ** 3 - 0.3 ** 3) * 1e-15
    v_nuc = 4.0 / 3.0 * math.pi * 0.3 ** 3 * 1e-15
    want = {"K": round(2.0e-6 * model.N_AVOGADRO * v_cyt), "S": round(8.0e-6 * model.N_AVOGADRO * v_cyt),
            "pS_n": round(3.0e-6 * model.N_AVOGADRO * v_nuc), "GENE": 2}
    got = {m.species[r.species].name: r.count for r in m.seed_records}
    assert got == want and want["pS_n"] == 204
    # translocation -> twin species and the per-contact threshold, both directions; mRNA export is one-way
    assert (m.species[ix["pS"]].cross_to, m.species[ix["pS_n"]].cross_to) == (ix["pS_n"], ix["pS"])
    assert m.species[ix["pS"]].cross_thr == model.prob_to_thr(0.05) == 214748365
    assert m.species[ix["mRNA_n"]].cross_to == ix["mRNA_c"] and m.species[ix["mRNA_c"]].cross_to == model.NONE16
    # expressor -> BIRTH with 1 - exp(-rate dt), before the consuming channels; degradation -> DEGRADE last
    g = m.species[ix["GENE:pS"]].channels
    assert [c.kind for c in g] == [model.CH_BIRTH, model.CH_RELEASE]
    assert g[0].prod1 == ix["mRNA_n"] and g[0].thr == model.prob_to_thr(1 - math.exp(-20_000.0 * 10e-6))
    assert (g[1].prod0, g[1].prod1) == (ix["GENE"], ix["pS_n"])
    r = m.species[ix["mRNA_c"]].channels
    assert [c.kind for c in r] == [model.CH_BIRTH, model.CH_DEGRADE] and r[1].thr == model.prob_to_thr(1 - math.exp(-5.0 * 10e-6))
    assert m.species[ix["GENE"]].sigma_class == 0 and m.species[ix["GENE:pS"]].sigma_class == 0        # immobile loci
    assert m.species[ix["pS"]].sigma_class == m.species[ix["S"]].sigma_class != 0
    import paper_2606_14603_b200 as pkg
    assert pkg.check_config(m) is None                                  # the compiled tables pass the library's checker


def test_checker_reports_compartment_mismatches():
    s = nuclear_spec(); s["molecules"][4]["interactions"][0]["partner"] = "K"          # nuclear pS_n binding cytosolic K
    assert any("partner K is localised in the cytosol, not the nucleus" in f for f in compiler.check(s))
    s = nuclear_spec(); s["molecules"][3]["translocation"]["to"] = "S"                  # twin in the same compartment
    assert any("translocation target S is localised in the same compartment" in f for f in compiler.check(s))
    s = nuclear_spec(); s["molecules"][8]["expression"]["product"] = "mRNA_n"           # cytosolic expressor, nuclear product
    assert any("expressed product mRNA_n is localised in the nucleus, not the cytosol" in f for f in compiler.check(s))
    s = nuclear_spec(); s["molecules"][6]["release"]["products"] = ["GENE", "pS"]       # nuclear complex releasing into the cytosol
    assert any("release product pS is localised in the cytosol, not the nucleus" in f for f in compiler.check(s))
    s = nuclear_spec(); del s["cell"]; s["volume_l"] = 1e-15                            # nucleus without a cell geometry
    assert any("needs a cell geometry with a nucleus" in f for f in compiler.check(s))
    s = nuclear_spec(); s["cell"]["nucleus_radius_um"] = 0.7
    assert any("nucleus_radius_um < radius_um" in f for f in compiler.check(s))
    s = nuclear_spec(); s["molecules"][3]["translocation"]["to"] = "nowhere"
    assert any("unknown molecule 'nowhere'" in f for f in compiler.check(s))


def test_compartmentalised_model_runs_on_the_oracle():
    from oracle.binding import Oracle

    m = compiler.compile_model(nuclear_spec(n_steps=300), cell_size=512)
    o = Oracle(m); o.seed_population(); o.step(300)
    a = o.read_agents()
    c = o.read_counts()[:, 0, :].astype(np.int64)
    ix = {s.name: i for i, s in enumerate(m.species)}
    comp = np.array([s.compartment for s in m.species])[a["species"]]
    r2 = sum((a[k].astype(np.int64) - 6000) ** 2 for k in "xyz")
    assert ((r2[comp == 0] > 3000 ** 2) & (r2[comp == 0] <= 6000 ** 2)).all() and (r2[comp == 1] <= 3000 ** 2).all()
    assert (c[:, ix["GENE"]] + c[:, ix["GENE:pS"]] == 2).all()                            # the two loci
    assert (c[:, ix["K"]] + c[:, ix["K:S"]] == c[0, ix["K"]]).all()                       # kinase moiety
    assert c[:, ix["pS"]].max() > 0 and c[:, ix["GENE:pS"]].max() > 0 and c[:, ix["mRNA_n"]].max() > 0


def test_shipped_example_model_files_compile_and_pass_the_library_checker():
    import os

    import paper_2606_14603_b200 as pkg

    d = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "workloads", "examples")
    for name, n_species in (("toy_cube.json", 3), ("nuclear_cell.json", 10)):
        text = open(os.path.join(d, name)).read()
        assert compiler.check(json.loads(text)) == []
        m = compiler.compile_model(text)
        assert len(m.species) == n_species and m.n_agents0 > 0 and pkg.check_config(m) is None
