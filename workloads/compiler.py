"""Model compiler: a model in PHYSICAL units (the paper's JSON model file) -> the integer tables the
step engine takes.  Host side only, runs once per model; no step arithmetic lives here.

What the paper states and what is chosen here (reading S26):
* a molecule is a sphere whose radius follows from its molecular weight.  The paper gives no
  formula; the minimal radius of a globular protein, r = 0.066 nm * MW[Da]^(1/3) (Erickson 2009), is used;
* its diffusion coefficient follows from Stokes-Einstein: D = k_B T / (6 pi eta r);
* product release is timed by the turnover number k_cat: per-step probability 1 - exp(-k_cat dt);
* species carry an initial concentration and a localisation; count = c * N_A * V;
* the consistency checker: reciprocal interaction definitions, every referenced molecule exists,
  molecular weights are plausible, volume and concentrations are compatible;
* localisation ("cytosolic or nuclear"): with a `cell` geometry (outer radius + nucleus radius,
  PAPER.md:153) a molecule lives in the cytosol (the shell) or in the nucleus; its count is its concentration times
  the volume of ITS compartment; `translocation` names its twin species in the other compartment and the crossing
  probability per membrane contact ("migrate between compartments at translocation rates"; reading
  S7); `expression` makes it an expressor that emits a product at a fixed rate = a BIRTH channel
  with probability 1 - exp(-rate dt); `degradation_per_s` = a DEGRADE channel.  The checker also
  reports partners, complexes and products that live in another compartment than the molecule that names them.
"""
import json
import math

from .model import (CH_BIRTH, CH_DEGRADE, CH_RELEASE, N_AVOGADRO, SHAPE_CUBE, SHAPE_SPHERE, Channel, Compartment, Model,
                    Reaction, SeedRecord, Species, prob_to_thr, sigma_units, stack_tables)

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


def compartment_volumes_l(spec: dict) -> dict:
    """Volume in litres of the compartment each localisation names: the whole cube, or shell / nucleus of a cell."""
    cell = spec.get("cell")
    if cell is None:
        return {"cytosol": spec.get("volume_l", 0.0)}
    r, rn = cell.get("radius_um", 0.0), cell.get("nucleus_radius_um", 0.0)
    f = 4.0 / 3.0 * math.pi * 1e-15
    return {"cytosol": f * (r ** 3 - rn ** 3), "nucleus": f * rn ** 3}


def check(spec: dict) -> list:
    """Returns the list of findings (empty = consistent)."""
    out = []
    names = [m["name"] for m in spec.get("molecules", [])]
    if len(set(names)) != len(names):
        out.append("duplicate molecule names")
    known = set(names)
    cell = spec.get("cell")
    vols = compartment_volumes_l(spec)
    if cell is not None:
        if not (0.0 < cell.get("nucleus_radius_um", 0.0) < cell.get("radius_um", 0.0)):
            out.append("cell: need 0 < nucleus_radius_um < radius_um")
    elif not spec.get("volume_l", 0.0) > 0.0:
        out.append("volume_l must be positive")
    loc = {m["name"]: m.get("localisation", "cytosol") for m in spec.get("molecules", [])}
    for m in spec.get("molecules", []):
        if loc[m["name"]] not in ("cytosol", "nucleus") or (cell is None and loc[m["name"]] != "cytosol"):
            out.append(f"{m['name']}: localisation {loc[m['name']]!r} needs a cell geometry with a nucleus")
            continue
        vol = vols.get(loc[m["name"]], 0.0)
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
                elif loc[it[key]] != loc[m["name"]]:
                    out.append(f"{m['name']}: {key} {it[key]} is localised in the {loc[it[key]]}, not the {loc[m['name']]}")
            p = next((q for q in spec["molecules"] if q["name"] == it.get("partner")), None)
            if p is not None and not any(r.get("partner") == m["name"] and r.get("complex") == it.get("complex")
                                         for r in p.get("interactions", [])):
                out.append(f"{m['name']} + {it['partner']}: no reciprocal interaction on {it['partner']}")
        rel = m.get("release")
        if rel:
            for pr in rel.get("products", []):
                if pr not in known:
                    out.append(f"{m['name']}: release refers to unknown molecule {pr!r}")
                elif loc[pr] != loc[m["name"]]:
                    out.append(f"{m['name']}: release product {pr} is localised in the {loc[pr]}, not the {loc[m['name']]}")
            if len(rel.get("products", [])) != 2:
                out.append(f"{m['name']}: a release needs exactly two products")
        tr = m.get("translocation")
        if tr:
            if tr.get("to") not in known:
                out.append(f"{m['name']}: translocation refers to unknown molecule {tr.get('to')!r}")
            elif loc[tr["to"]] == loc[m["name"]]:
                out.append(f"{m['name']}: translocation target {tr['to']} is localised in the same compartment")
            if not 0.0 <= tr.get("prob_per_contact", -1.0) <= 1.0:
                out.append(f"{m['name']}: translocation needs prob_per_contact in [0, 1]")
        ex = m.get("expression")
        if ex:
            if ex.get("product") not in known:
                out.append(f"{m['name']}: expression refers to unknown molecule {ex.get('product')!r}")
            elif loc[ex["product"]] != loc[m["name"]]:
                out.append(f"{m['name']}: expressed product {ex['product']} is localised in the {loc[ex['product']]}, "
                           f"not the {loc[m['name']]}")
            if not ex.get("rate_per_s", 0.0) > 0.0:
                out.append(f"{m['name']}: expression needs a positive rate_per_s")
        if m.get("degradation_per_s", 0.0) < 0.0:
            out.append(f"{m['name']}: negative degradation rate")
    return out


def compile_model(spec, cell_size: int = 512, table_bits: int = 12, capacity_factor: float = 1.6) -> Model:
    """spec: dict or JSON text.  Geometry: one reflective cube of `volume_l` [CFG 0-shaped], or with `cell`
    {radius_um, nucleus_radius_um} a cytosol shell around a concentric nucleus [CFG 3-shaped].  Every molecule gets
    its radius, D and sigma-class from its molecular weight (`immobile`: class 0); interactions -> reactions (anchor =
    the molecule that lists the interaction first); channels, in this order (reading S13: the lowest consuming
    channel that fires applies): expression -> BIRTH, release -> RELEASE (probability from k_cat),
    degradation_per_s -> DEGRADE; translocation -> cross_to / cross_thr."""
    if isinstance(spec, str):
        spec = json.loads(spec)
    bad = check(spec)
    if bad:
        raise ModelError("; ".join(bad))
    dt_us = float(spec["dt_us"])
    temp, eta = spec.get("temperature_k", 310.15), spec.get("viscosity_pa_s", 6.913e-4)
    mols = spec["molecules"]
    ix = {m["name"]: i for i, m in enumerate(mols)}
    cell = spec.get("cell")
    comp_of = {"cytosol": 0, "nucleus": 1}
    vols = compartment_volumes_l(spec)
    # sigma classes: one per distinct sigma (class 0 = immobile is implicit in stack_tables)
    sig = [0.0 if m.get("immobile") else sigma_units(stokes_einstein_um2_s(radius_nm(m["mw_da"]), temp, eta), dt_us)
           for m in mols]
    classes = sorted(set(round(s, 6) for s in sig if s > 0.0))
    species = []
    for m, s in zip(mols, sig):
        ch = []
        if m.get("expression"):
            ch.append(Channel(CH_BIRTH, prob_to_thr(kcat_to_prob(m["expression"]["rate_per_s"], dt_us)),
                              prod1=ix[m["expression"]["product"]]))
        if m.get("release"):
            a, b = (ix[p] for p in m["release"]["products"])
            ch.append(Channel(CH_RELEASE, prob_to_thr(kcat_to_prob(m["release"]["kcat_per_s"], dt_us)), a, b))
        if m.get("degradation_per_s", 0.0) > 0.0:
            ch.append(Channel(CH_DEGRADE, prob_to_thr(kcat_to_prob(m["degradation_per_s"], dt_us))))
        sp = Species(m["name"], classes.index(round(s, 6)) + 1 if s > 0.0 else 0,
                     comp_of[m.get("localisation", "cytosol")], channels=ch)
        if m.get("translocation"):
            sp.cross_to = ix[m["translocation"]["to"]]
            sp.cross_thr = prob_to_thr(m["translocation"]["prob_per_contact"])
        species.append(sp)
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
    recs = [SeedRecord(ix[m["name"]], count_from_concentration(m.get("concentration_molar", 0.0),
                                                               vols[m.get("localisation", "cytosol")]))
            for m in mols if m.get("concentration_molar", 0.0) > 0.0]
    recs += [SeedRecord(ix[m["name"]], int(m["count"])) for m in mols if m.get("count", 0) > 0]   # e.g. two gene loci
    if cell is None:
        edge_units = int(round((spec["volume_l"] * 1e15) ** (1.0 / 3.0) * 1e4))      # 1 L = 1e15 um^3, 1 um = 1e4 units
        comps, extent, vol_um3 = [Compartment(SHAPE_CUBE, L=edge_units)], (edge_units,) * 3, spec["volume_l"] * 1e15
    else:
        R, Rn = int(round(cell["radius_um"] * 1e4)), int(round(cell["nucleus_radius_um"] * 1e4))
        comps = [Compartment(SHAPE_SPHERE, R, R, R, r_out=R, r_in=Rn), Compartment(SHAPE_SPHERE, R, R, R, r_out=Rn)]
        extent, vol_um3 = (2 * R + 1,) * 3, (vols["cytosol"] + vols["nucleus"]) * 1e15
    model = Model(name=spec.get("name", "compiled"), species=species, reactions=reactions, compartments=comps,
                  table_bits=table_bits, tables=stack_tables(classes, table_bits), extent=extent,
                  seed=int(spec.get("seed", 1)), place_seed=int(spec.get("seed", 1)), seed_records=recs,
                  n_steps=int(spec.get("n_steps", 100)), cell_size=cell_size, dt_us=dt_us, volume_um3=vol_um3)
    n0 = sum(r.count for r in recs)
    model.capacity = int(n0 * capacity_factor) + 4096
    return model.finalize()
