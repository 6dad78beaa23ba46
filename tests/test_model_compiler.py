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
