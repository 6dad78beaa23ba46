"""Model compiler: a model in PHYSICAL units (the paper's JSON model file) -> the integer tables the
step engine takes.  Host side only, runs once per model; no step arithmetic lives here.

What the paper states and what is chosen here (reading S26):
* a molecule is a sphere whose radius follows from its molecular weight.  The paper gives no
  formula; the minimal radius of a globular protein, r = 0.066 nm * MW[Da]^(1/3) (Erickson 2009), is used;
* its diffusion coefficient follows from Stokes-Einstein: D = k_B T / (6 pi eta r);
* product release is timed by the turnover number k_cat: per-step probability 1 - exp(-k_cat dt);
* species carry an initial concentration and a localisation; count = c * N_A * V;
* the consistency checker: reciprocal interaction definitions, every referenced molecule exists,
  molecular weights are plausible, volume and concentrations are compatible.
"""
import json
import math

from .model import (CH_RELEASE, N_AVOGADRO, SHAPE_CUBE, Channel, Compartment, Model, Reaction, SeedRecord, Species,
                    prob_to_thr, sigma_units, stack_tables)

K_BOLTZMANN = 1.380649e-23          # J/K (exact, SI 2019)


class ModelError(ValueError):
    """The consistency checker's findings, one line each."""


def radius_nm(mw_da: float) -> float:
    return 0.066 * mw_da ** (1.0 / 3.0)


def stokes_einstein_um2_s(radius_nm_: float, temperature_k: float = 310.15, viscosity_pa_s: float = 6.913e-4) -> float:
    """D = k_B T / (6 pi eta r) in um^2/s (defaults: 37 C, water)."""
    d_m2_s = K_BOLTZMANN * temperature_k / (6.0 * math.pi * viscosity_pa_s * radius_nm_ * 1e-9)
    return d_m2_s * 1e12


def kcat_to_prob(kcat_per_s: float, dt_us: float) -> float:
    return 1.0 - math.exp(-kcat_per_s * dt_us * 1e-6)


def count_from_concentration(c_molar: float, volume_l: float) -> int:
    return int(round(c_molar * N_AVOGADRO * volume_l))


def check(spec: dict) -> list:
    """Returns the list of findings (empty = consistent)."""
    out = []
    names = [m["name"] for m in spec.get("molecules", [])]
    if len(set(names)) != len(names):
        out.append("duplicate molecule names")
    known = set(names)
    vol = spec.get("volume_l", 0.0)
    if not vol > 0.0:
        out.append("volume_l must be positive")
    for m in spec.get("molecules", []):
        mw = m.get("mw_da", 0.0)
        if not 50.0 <= mw <= 5e6:
            out.append(f"{m['name']}: molecular weight {mw} Da is not plausible")
        c = m.get("concentration_molar", 0.0)
        if c < 0.0:
            out.append(f"{m['name']}: negative concentration")
        elif c > 0.0 and vol > 0.0 and count_from_concentration(c, vol) < 1:
            out.append(f"{m['name']}: {c} M in {vol} L is less than one molecule")
        for it in m.get("interactions", []):
            for key in ("partner", "complex"):
                if it.get(key) not in known:
                    out.append(f"{m['name']}: interaction refers to unknown molecule {it.get(key)!r}")
            p = next((q for q in spec["molecules"] if q["name"] == it.get("partner")), None)
            if p is not None and not any(r.get("partner") == m["name"] and r.get("complex") == it.get("complex")
                                         for r in p.get("interactions", [])):
                out.append(f"{m['name']} + {it['partner']}: no reciprocal interaction on {it['partner']}")
        rel = m.get("release")
        if rel:
            for pr in rel.get("products", []):
                if pr not in known:
                    out.append(f"{m['name']}: release refers to unknown molecule {pr!r}")
            if len(rel.get("products", [])) != 2:
                out.append(f"{m['name']}: a release needs exactly two products")
    return out


def compile_model(spec, cell_size: int = 512, table_bits: int = 12, capacity_factor: float = 1.6) -> Model:
    """spec: dict or JSON text.  One reflective cube of the given volume [CFG 0-shaped]; every molecule gets its
    radius, D and sigma-class from its molecular weight; interactions -> reactions (anchor = the molecule that
    lists the interaction first); release -> a RELEASE channel with probability from k_cat."""
    if isinstance(spec, str):
        spec = json.loads(spec)
    bad = check(spec)
    if bad:
        raise ModelError("; ".join(bad))
    dt_us = float(spec["dt_us"])
    temp, eta = spec.get("temperature_k", 310.15), spec.get("viscosity_pa_s", 6.913e-4)
    mols = spec["molecules"]
    ix = {m["name"]: i for i, m in enumerate(mols)}
    # sigma classes: one per distinct sigma (class 0 = immobile is implicit in stack_tables)
    sig = [sigma_units(stokes_einstein_um2_s(radius_nm(m["mw_da"]), temp, eta), dt_us) for m in mols]
    classes = sorted(set(round(s, 6) for s in sig))
    species = []
    for m, s in zip(mols, sig):
        ch = []
        if m.get("release"):
            a, b = (ix[p] for p in m["release"]["products"])
            ch.append(Channel(CH_RELEASE, prob_to_thr(kcat_to_prob(m["release"]["kcat_per_s"], dt_us)), a, b))
        species.append(Species(m["name"], classes.index(round(s, 6)) + 1, channels=ch))
    reactions, seen = [], set()
    for m in mols:
        for it in m.get("interactions", []):
            pair = frozenset((m["name"], it["partner"]))
            if pair in seen:
                continue
            seen.add(pair)
            r_units = int(round(it["radius_nm"] * 10.0))
            reactions.append(Reaction(ix[m["name"]], ix[it["partner"]], ix[it["complex"]], r_units * r_units,
                                      prob_to_thr(it["p_bind"])))
    edge_units = int(round((spec["volume_l"] * 1e15) ** (1.0 / 3.0) * 1e4))      # 1 L = 1e15 um^3, 1 um = 1e4 units
    recs = [SeedRecord(ix[m["name"]], count_from_concentration(m.get("concentration_molar", 0.0), spec["volume_l"]))
            for m in mols if m.get("concentration_molar", 0.0) > 0.0]
    model = Model(name=spec.get("name", "compiled"), species=species, reactions=reactions,
                  compartments=[Compartment(SHAPE_CUBE, L=edge_units)], table_bits=table_bits,
                  tables=stack_tables(classes, table_bits), extent=(edge_units,) * 3, seed=int(spec.get("seed", 1)),
                  place_seed=int(spec.get("seed", 1)), seed_records=recs, n_steps=int(spec.get("n_steps", 100)),
                  cell_size=cell_size, dt_us=dt_us, volume_um3=spec["volume_l"] * 1e15)
    n0 = sum(r.count for r in recs)
    model.capacity = int(n0 * capacity_factor) + 4096
    return model.finalize()
