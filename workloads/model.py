"""Neutral, integer-only description of a molecule-agent model.

This module is the *input side* shared by the oracle tests, the CUDA binding,
bench.py and smoke(): it turns physical units (um^2/s, us, nm, probabilities)
into the integer tables that both implementations take as DATA (DESIGN.md
readings S3, S4).  It contains none of the step arithmetic (no Philox, no move,
no binding, no reactions): neither `oracle/` nor the CUDA path is imported here
and each of them marshals a `Model` into its own C structs.

Units: positions are int32 in 0.1 nm units [north_star (1)], so 1 nm = 10 units
and 1 um = 10,000 units.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Sequence, Tuple

import numpy as np

NONE16 = 0xFFFF  # "no species" / DEAD marker

# unimolecular channel kinds (DESIGN.md step spec, phase 3)
CH_NONE, CH_BIRTH, CH_RELEASE, CH_CONVERT, CH_DEGRADE, CH_DELAYED_BIRTH = 0, 1, 2, 3, 4, 5
# compartment shapes
SHAPE_CUBE, SHAPE_SPHERE = 0, 1  # SPHERE with r_in >= 0 is a shell

UNITS_PER_NM = 10
UNITS_PER_UM = 10_000
MAX_CHANNELS = 4


def prob_to_thr(p: float) -> int:
    """Probability -> uint32 threshold (reading S4): min(floor(p*2^32+0.5), 2^32-1)."""
    if not (0.0 <= p <= 1.0):
        raise ValueError("probability outside [0,1]")
    return min(int(math.floor(p * 4294967296.0 + 0.5)), 0xFFFFFFFF)


def sigma_units(D_um2_s: float, dt_us: float) -> float:
    """sigma = sqrt(2 D dt) per axis [north_star (2)], in 0.1 nm units."""
    return math.sqrt(2.0 * D_um2_s * dt_us * 1e-6) * UNITS_PER_UM


def gaussian_table(sigma: float, bits: int) -> np.ndarray:
    """Integer inverse-CDF table of the discretised Gaussian (reading S3).

    entry k = round_half_away(sigma * Phi^-1((k + 0.5) / 2^bits)), int16.
    """
    from scipy.special import ndtri

    n = 1 << bits
    q = sigma * ndtri((np.arange(n, dtype=np.float64) + 0.5) / n)
    t = np.sign(q) * np.floor(np.abs(q) + 0.5)
    if np.max(np.abs(t)) > 32767:
        raise ValueError("sigma too large for int16 table")
    return t.astype(np.int16)


@dataclass
class Channel:
    kind: int
    thr: int = 0          # uint32 threshold; for DELAYED_BIRTH: delay in steps (>= 1)
    prod0: int = NONE16   # species the parent becomes (RELEASE / CONVERT)
    prod1: int = NONE16   # species of the newborn (BIRTH / RELEASE / DELAYED_BIRTH)
    rule: int = 0         # t_first slot (BIRTH with marks_first, DELAYED_BIRTH)
    marks_first: bool = False


@dataclass
class Species:
    name: str
    sigma_class: int = 0          # 0 = immobile
    compartment: int = 0
    cross_to: int = NONE16        # twin species in the adjacent compartment
    cross_thr: int = 0
    channels: List[Channel] = field(default_factory=list)


@dataclass
class Reaction:
    a: int        # anchor reactant: keeps id and position, becomes the complex (S10)
    b: int
    cplx: int
    r2: int       # interaction radius squared, units^2
    thr: int      # pair-draw threshold


@dataclass
class Compartment:
    shape: int
    cx: int = 0
    cy: int = 0
    cz: int = 0
    L: int = 0        # cube edge: lattice points 0..L-1 (local coordinates)
    r_out: int = 0    # sphere: |p-c|^2 <= r_out^2
    r_in: int = -1    # shell: additionally |p-c|^2 > r_in^2 ; -1 = no hole


@dataclass
class SeedRecord:
    species: int
    count: int
    replica: int = 0


@dataclass
class Model:
    name: str
    species: List[Species]
    reactions: List[Reaction]
    compartments: List[Compartment]
    table_bits: int
    tables: np.ndarray            # int16 [n_sigma_classes, 2^table_bits]; row 0 unused (immobile)
    extent: Tuple[int, int, int]  # world bounding box: 0 <= p < extent
    seed: int                     # u64 simulation seed (Philox key)
    place_seed: int               # u64 placement seed
    seed_records: List[SeedRecord]
    n_steps: int                  # nominal run length of the workload
    cell_size: int                # spatial-hash cell edge (tuning hint, >= max R)
    n_replicas: int = 1
    stride_shift: int = 31        # replica = x >> stride_shift
    n_rules: int = 1
    capacity: int = 0             # max agent slots
    id_capacity: int = 0          # max ids ever issued
    counts_rows: int = 0
    dt_us: float = 1.0
    volume_um3: float = 0.0       # per replica, for derived concentration curves

    @property
    def n_species(self) -> int:
        return len(self.species)

    @property
    def n_agents0(self) -> int:
        return sum(r.count for r in self.seed_records)

    def species_index(self, name: str) -> int:
        for i, s in enumerate(self.species):
            if s.name == name:
                return i
        raise KeyError(name)

    def finalize(self, steps_headroom: int | None = None) -> "Model":
        """Fill capacity / id_capacity / counts_rows defaults from the seeded population."""
        n0 = self.n_agents0
        steps = self.n_steps if steps_headroom is None else steps_headroom
        if self.capacity == 0:
            self.capacity = int(n0 * 1.25) + 4096
        if self.id_capacity == 0:
            self.id_capacity = int(n0 * 2) + 65536
        if self.counts_rows == 0:
            self.counts_rows = steps + 1
        return self


def stack_tables(sigmas: Sequence[float], bits: int) -> np.ndarray:
    """Row 0 = immobile class (zeros); row c = table for sigmas[c-1]."""
    rows = [np.zeros(1 << bits, dtype=np.int16)]
    rows += [gaussian_table(s, bits) for s in sigmas]
    return np.stack(rows)


N_AVOGADRO = 6.02214076e23


def concentration_molar(counts: np.ndarray, volume_um3: float) -> np.ndarray:
    """Derived concentration curve c = n / (N_A * V) in mol/L, float64."""
    litres = volume_um3 * 1e-15
    return np.asarray(counts, dtype=np.float64) / (N_AVOGADRO * litres)
