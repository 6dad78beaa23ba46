"""ctypes binding of oracle/liboracle.so.  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs import this.  It marshals a neutral `workloads.Model` into the oracle's own C
structs (oracle/oracle.h); it shares nothing with the CUDA binding.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

NOPROP = 0xFFFFFFFF
MODE_GRID, MODE_BRUTE = 0, 1
E_INVAL, E_CAPACITY, E_IDSPACE = -1, -2, -3


class _Channel(C.Structure):
    _fields_ = [("kind", C.c_uint32), ("thr", C.c_uint32), ("prod0", C.c_uint16),
                ("prod1", C.c_uint16), ("rule", C.c_uint16), ("marks_first", C.c_uint16)]


class _Species(C.Structure):
    _fields_ = [("sigma_class", C.c_uint16), ("compartment", C.c_uint16), ("cross_to", C.c_uint16),
                ("n_channels", C.c_uint16), ("cross_thr", C.c_uint32), ("ch", _Channel * 4)]


class _Reaction(C.Structure):
    _fields_ = [("a", C.c_uint16), ("b", C.c_uint16), ("cplx", C.c_uint16), ("pad", C.c_uint16),
                ("r2", C.c_uint32), ("thr", C.c_uint32)]


class _Compartment(C.Structure):
    _fields_ = [("shape", C.c_uint32), ("cx", C.c_int32), ("cy", C.c_int32), ("cz", C.c_int32),
                ("L", C.c_int32), ("r_out", C.c_int32), ("r_in", C.c_int32)]


class _SeedRec(C.Structure):
    _fields_ = [("species", C.c_uint16), ("replica", C.c_uint16), ("count", C.c_uint32)]


class _Config(C.Structure):
    _fields_ = [("n_species", C.c_uint32), ("n_reactions", C.c_uint32), ("n_compartments", C.c_uint32),
                ("n_sigma_classes", C.c_uint32), ("table_bits", C.c_uint32), ("n_rules", C.c_uint32),
                ("n_replicas", C.c_uint32), ("stride_shift", C.c_uint32), ("extent", C.c_int32 * 3),
                ("cell_size", C.c_uint32), ("seed", C.c_uint64), ("capacity", C.c_uint32),
                ("id_capacity", C.c_uint32), ("counts_rows", C.c_uint32), ("pad", C.c_uint32),
                ("species", C.POINTER(_Species)), ("reactions", C.POINTER(_Reaction)),
                ("compartments", C.POINTER(_Compartment)), ("tables", C.POINTER(C.c_int16))]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp, u32, u64 = C.c_void_p, C.c_uint32, C.c_uint64
        P = C.POINTER
        L.oracle_create.argtypes = [P(_Config), P(vp)]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_destroy.restype = None
        L.oracle_set_mode.argtypes = [vp, C.c_int]
        L.oracle_seed_population.argtypes = [vp, P(_SeedRec), u32, u64]
        L.oracle_step.argtypes = [vp, u32]
        L.oracle_read_counts.argtypes = [vp, u32, u32, vp]
        L.oracle_read_agents.argtypes = [vp, u32, vp, vp, vp, vp, vp, P(u32)]
        L.oracle_load_agents.argtypes = [vp, u32, vp, vp, vp, vp, vp, u32, u32]
        L.oracle_info.argtypes = [vp, P(u32), P(u32), P(u32), P(u32)]
        L.oracle_read_checksum.argtypes = [vp, P(u64)]
        L.oracle_read_t_first.argtypes = [vp, u32, vp]
        L.oracle_load_t_first.argtypes = [vp, u32, vp]
        L.oracle_philox4x32_10.argtypes = [vp, vp, vp]
        L.oracle_philox4x32_10.restype = None
        L.oracle_debug_move_only.argtypes = [vp]
        L.oracle_debug_proposals.argtypes = [vp, C.c_int, vp]
        L.oracle_debug_pairs.argtypes = [vp, C.c_int, u32, vp, P(u32)]
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__(f"oracle error {code}")
        self.code = code


def _chk(code):
    if code != 0:
        raise OracleError(code)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def philox(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
    return out


class Oracle:
    """One population driven through the oracle's C ABI (same call names as the product's)."""

    def __init__(self, model, cell_size=None, seed=None, mode=MODE_GRID):
        m = model
        self.model = m
        sp = (_Species * len(m.species))()
        for i, s in enumerate(m.species):
            sp[i].sigma_class, sp[i].compartment = s.sigma_class, s.compartment
            sp[i].cross_to, sp[i].cross_thr, sp[i].n_channels = s.cross_to, s.cross_thr, len(s.channels)
            for k, ch in enumerate(s.channels):
                c = sp[i].ch[k]
                c.kind, c.thr, c.prod0, c.prod1 = ch.kind, ch.thr, ch.prod0, ch.prod1
                c.rule, c.marks_first = ch.rule, int(ch.marks_first)
        rx = (_Reaction * max(1, len(m.reactions)))()
        for i, r in enumerate(m.reactions):
            rx[i].a, rx[i].b, rx[i].cplx, rx[i].r2, rx[i].thr = r.a, r.b, r.cplx, r.r2, r.thr
        cp = (_Compartment * len(m.compartments))()
        for i, c in enumerate(m.compartments):
            cp[i].shape, cp[i].cx, cp[i].cy, cp[i].cz = c.shape, c.cx, c.cy, c.cz
            cp[i].L, cp[i].r_out, cp[i].r_in = c.L, c.r_out, c.r_in
        tab = np.ascontiguousarray(m.tables, dtype=np.int16)
        cfg = _Config()
        cfg.n_species, cfg.n_reactions, cfg.n_compartments = len(m.species), len(m.reactions), len(m.compartments)
        cfg.n_sigma_classes, cfg.table_bits, cfg.n_rules = tab.shape[0], m.table_bits, m.n_rules
        cfg.n_replicas, cfg.stride_shift = m.n_replicas, m.stride_shift
        cfg.extent = (C.c_int32 * 3)(*m.extent)
        cfg.cell_size = m.cell_size if cell_size is None else cell_size
        cfg.seed = m.seed if seed is None else seed
        cfg.capacity, cfg.id_capacity, cfg.counts_rows = m.capacity, m.id_capacity, m.counts_rows
        cfg.species, cfg.reactions, cfg.compartments = sp, rx, cp
        cfg.tables = tab.ctypes.data_as(C.POINTER(C.c_int16))
        self._keep = (sp, rx, cp, tab)
        h = C.c_void_p()
        _chk(lib().oracle_create(C.byref(cfg), C.byref(h)))
        self._h = h
        self.row_width = m.n_replicas * len(m.species)
        if mode != MODE_GRID:
            self.set_mode(mode)

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    __del__ = close

    def set_mode(self, mode):
        _chk(lib().oracle_set_mode(self._h, mode))

    def seed_population(self, records=None, place_seed=None):
        records = self.model.seed_records if records is None else records
        place_seed = self.model.place_seed if place_seed is None else place_seed
        recs = (_SeedRec * max(1, len(records)))()
        for i, r in enumerate(records):
            recs[i].species, recs[i].replica, recs[i].count = r.species, r.replica, r.count
        _chk(lib().oracle_seed_population(self._h, recs, len(records), place_seed))

    def step(self, n=1):
        _chk(lib().oracle_step(self._h, n))

    def info(self):
        a, b, c, d = C.c_uint32(), C.c_uint32(), C.c_uint32(), C.c_uint32()
        _chk(lib().oracle_info(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(d)))
        return {"n_live": a.value, "step": b.value, "next_id": c.value, "t_first0": d.value}

    def read_counts(self, first_row=0, n_rows=None):
        if n_rows is None:
            n_rows = self.info()["step"] + 1 - first_row
        out = np.zeros((n_rows, self.model.n_replicas, len(self.model.species)), dtype=np.uint32)
        _chk(lib().oracle_read_counts(self._h, first_row, n_rows, _ptr(out)))
        return out

    def read_agents(self):
        n = self.info()["n_live"]
        x, y, z = (np.zeros(n, dtype=np.int32) for _ in range(3))
        s = np.zeros(n, dtype=np.uint16)
        i = np.zeros(n, dtype=np.uint32)
        k = C.c_uint32()
        _chk(lib().oracle_read_agents(self._h, n, _ptr(x), _ptr(y), _ptr(z), _ptr(s), _ptr(i), C.byref(k)))
        return {"x": x, "y": y, "z": z, "species": s, "id": i}

    def load_agents(self, x, y, z, species, id, step=0, next_id=None):
        x, y, z = (np.ascontiguousarray(a, dtype=np.int32) for a in (x, y, z))
        s = np.ascontiguousarray(species, dtype=np.uint16)
        i = np.ascontiguousarray(id, dtype=np.uint32)
        if next_id is None:
            next_id = int(i.max()) + 1 if len(i) else 0
        _chk(lib().oracle_load_agents(self._h, len(x), _ptr(x), _ptr(y), _ptr(z), _ptr(s), _ptr(i), step, next_id))

    def read_checksum(self):
        v = C.c_uint64()
        _chk(lib().oracle_read_checksum(self._h, C.byref(v)))
        return v.value

    def read_t_first(self):
        out = np.zeros(max(1, self.model.n_rules), dtype=np.uint32)
        if self.model.n_rules:
            _chk(lib().oracle_read_t_first(self._h, self.model.n_rules, _ptr(out)))
        return out[: self.model.n_rules]

    def load_t_first(self, t_first):
        a = np.ascontiguousarray(t_first, dtype=np.uint32)
        _chk(lib().oracle_load_t_first(self._h, len(a), _ptr(a)))

    def debug_move_only(self):
        _chk(lib().oracle_debug_move_only(self._h))

    def debug_proposals(self, mode):
        out = np.zeros(self.info()["n_live"], dtype=np.uint32)
        _chk(lib().oracle_debug_proposals(self._h, mode, _ptr(out)))
        return out

    def debug_pairs(self, mode, cap=1 << 20):
        out = np.zeros((cap, 2), dtype=np.uint32)
        n = C.c_uint32()
        _chk(lib().oracle_debug_pairs(self._h, mode, cap, _ptr(out), C.byref(n)))
        return out[: n.value].copy()
