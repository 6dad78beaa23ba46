"""ctypes binding of libmolsim.so — same call names as include/molsim.h, marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
# MOLSIM_CHECKS=1 (tests only) loads the checked build, libmolsim_checked.so (build.py; device-side bound checks)
LIB_PATH = os.path.join(HERE, "libmolsim_checked.so" if os.environ.get("MOLSIM_CHECKS") == "1" else "libmolsim.so")
N_KERNELS = 10
E_INVAL, E_CAPACITY, E_IDSPACE, E_CUDA = -1, -2, -3, -4


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


EXPORTS = ["sim_workspace_bytes", "sim_create", "sim_seed_population", "sim_step", "sim_step_async",
           "sim_read_counts", "sim_read_agents", "sim_load_agents", "sim_info", "sim_debug_move_only",
           "sim_launch_count", "sim_profile_enable", "sim_kernel_times", "sim_kernel_name", "sim_destroy",
           "sim_strerror", "sim_last_cuda_error", "sim_debug_philox", "sim_monitor_eval", "sim_render",
           "sim_read_checksum", "sim_read_t_first", "sim_load_t_first", "sim_check_config"]

_lib = None


def load_library():
    """Loads libmolsim.so; raises (never falls back) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(nvcc, sm_100a). There is no CPU fallback.")
    _lib = declare_signatures(C.CDLL(LIB_PATH))
    return _lib


def declare_signatures(L):
    """ctypes argument / result types of every export of include/molsim.h on a loaded library."""
    vp, u32, u64, P = C.c_void_p, C.c_uint32, C.c_uint64, C.POINTER
    L.sim_workspace_bytes.argtypes = [P(_Config)]
    L.sim_workspace_bytes.restype = C.c_size_t
    L.sim_create.argtypes = [P(_Config), vp, C.c_size_t, vp, P(vp)]
    L.sim_seed_population.argtypes = [vp, P(_SeedRec), u32, u64]
    L.sim_step.argtypes = [vp, u32]
    L.sim_step_async.argtypes = [vp, u32]
    L.sim_read_counts.argtypes = [vp, u32, u32, vp]
    L.sim_read_agents.argtypes = [vp, u32, vp, vp, vp, vp, vp, P(u32)]
    L.sim_load_agents.argtypes = [vp, u32, vp, vp, vp, vp, vp, u32, u32]
    L.sim_info.argtypes = [vp, P(u32), P(u32), P(u32), P(u32)]
    L.sim_read_checksum.argtypes = [vp, P(C.c_uint64)]
    L.sim_read_t_first.argtypes = [vp, u32, vp]
    L.sim_load_t_first.argtypes = [vp, u32, vp]
    L.sim_check_config.argtypes = [P(_Config)]
    L.sim_check_config.restype = C.c_char_p
    L.sim_debug_move_only.argtypes = [vp]
    L.sim_launch_count.argtypes = [vp]
    L.sim_launch_count.restype = C.c_uint64
    L.sim_profile_enable.argtypes = [vp, C.c_int]
    L.sim_kernel_times.argtypes = [vp, vp, vp]
    L.sim_kernel_name.argtypes = [C.c_int]
    L.sim_kernel_name.restype = C.c_char_p
    L.sim_destroy.argtypes = [vp]
    L.sim_destroy.restype = None
    L.sim_strerror.argtypes = [C.c_int]
    L.sim_strerror.restype = C.c_char_p
    L.sim_last_cuda_error.argtypes = [vp]
    L.sim_last_cuda_error.restype = C.c_char_p
    L.sim_debug_philox.argtypes = [vp, vp, vp, u32, vp]
    L.sim_monitor_eval.argtypes = [vp, vp, u32, vp, vp, u32]
    L.sim_render.argtypes = [vp, vp, vp]
    return L


class _Monitor(C.Structure):
    _fields_ = [("replica", C.c_uint32), ("n_species", C.c_uint32), ("species", C.c_uint16 * 4),
                ("threshold", C.c_uint32), ("first_row", C.c_uint32), ("n_rows", C.c_uint32)]


class _MonitorResult(C.Structure):
    _fields_ = [("first_above", C.c_uint32), ("n_above", C.c_uint32), ("last_state", C.c_uint32),
                ("max_value", C.c_uint32), ("max_row", C.c_uint32), ("n_switches", C.c_uint32)]


class _View(C.Structure):
    _fields_ = [("replica", C.c_uint32), ("axis", C.c_uint32), ("u0", C.c_int32), ("v0", C.c_int32),
                ("eu", C.c_uint32), ("ev", C.c_uint32), ("width", C.c_uint32), ("height", C.c_uint32),
                ("gain", C.c_uint32), ("palette", (C.c_uint8 * 4) * 8)]


class SimError(RuntimeError):
    def __init__(self, code, detail=""):
        msg = load_library().sim_strerror(code).decode()
        super().__init__(f"molsim error {code}: {msg} {detail}")
        self.code = code


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def marshal_config(m, cell_size=None, seed=None):
    """workloads.Model -> sim_config_t (+ the ctypes objects that must stay alive)."""
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
    return cfg, (sp, rx, cp, tab)


def check_config(model, cell_size=None):
    """sim_check_config: None when the tables are valid, else the name of the first rule (V1-V7) that fails.  Host only."""
    cfg, keep = marshal_config(model, cell_size, None)
    why = load_library().sim_check_config(C.byref(cfg))
    return None if why is None else why.decode()


class Sim:
    """One population on one GPU.  Methods mirror the C ABI one to one."""

    def __init__(self, model, cell_size=None, seed=None, device="cuda:0", stream=None):
        import torch

        self._lib = load_library()
        self.model = model
        cfg, keep = marshal_config(model, cell_size, seed)
        nbytes = self._lib.sim_workspace_bytes(C.byref(cfg))
        if nbytes == 0:
            why = self._lib.sim_check_config(C.byref(cfg))
            raise SimError(E_INVAL, f"(sim_workspace_bytes: {why.decode() if why else 'cell grid too large'})")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        self._check(self._lib.sim_create(C.byref(cfg), C.c_void_p(base), nbytes,
                                         C.c_void_p(self.stream.cuda_stream), C.byref(h)))
        self._h = h
        self.workspace_bytes = nbytes

    def _check(self, code):
        if code != 0:
            detail = ""
            if code == E_CUDA and getattr(self, "_h", None):
                detail = self._lib.sim_last_cuda_error(self._h).decode()
            raise SimError(code, detail)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.sim_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def seed_population(self, records=None, place_seed=None):
        records = self.model.seed_records if records is None else records
        place_seed = self.model.place_seed if place_seed is None else place_seed
        recs = (_SeedRec * max(1, len(records)))()
        for i, r in enumerate(records):
            recs[i].species, recs[i].replica, recs[i].count = r.species, r.replica, r.count
        self._check(self._lib.sim_seed_population(self._h, recs, len(records), place_seed))

    def step(self, n=1):
        self._check(self._lib.sim_step(self._h, n))

    def step_async(self, n=1):
        self._check(self._lib.sim_step_async(self._h, n))

    def info(self):
        a, b, c, d = C.c_uint32(), C.c_uint32(), C.c_uint32(), C.c_uint32()
        self._check(self._lib.sim_info(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(d)))
        return {"n_live": a.value, "step": b.value, "next_id": c.value, "t_first0": d.value}

    def read_counts(self, first_row=0, n_rows=None):
        if n_rows is None:
            n_rows = self.info()["step"] + 1 - first_row
        out = np.zeros((n_rows, self.model.n_replicas, len(self.model.species)), dtype=np.uint32)
        self._check(self._lib.sim_read_counts(self._h, first_row, n_rows, _ptr(out)))
        return out

    def read_agents(self, cap=None):
        n = self.info()["n_live"] if cap is None else cap
        x, y, z = (np.zeros(n, dtype=np.int32) for _ in range(3))
        s = np.zeros(n, dtype=np.uint16)
        i = np.zeros(n, dtype=np.uint32)
        k = C.c_uint32()
        self._check(self._lib.sim_read_agents(self._h, n, _ptr(x), _ptr(y), _ptr(z), _ptr(s), _ptr(i), C.byref(k)))
        m = k.value
        return {"x": x[:m], "y": y[:m], "z": z[:m], "species": s[:m], "id": i[:m]}

    def load_agents(self, x, y, z, species, id, step=0, next_id=None):
        x, y, z = (np.ascontiguousarray(a, dtype=np.int32) for a in (x, y, z))
        s = np.ascontiguousarray(species, dtype=np.uint16)
        i = np.ascontiguousarray(id, dtype=np.uint32)
        if next_id is None:
            next_id = int(i.max()) + 1 if len(i) else 0
        self._check(self._lib.sim_load_agents(self._h, len(x), _ptr(x), _ptr(y), _ptr(z), _ptr(s), _ptr(i),
                                              step, next_id))

    def read_checksum(self):
        v = C.c_uint64()
        self._check(self._lib.sim_read_checksum(self._h, C.byref(v)))
        return v.value

    def read_t_first(self):
        out = np.zeros(max(1, self.model.n_rules), dtype=np.uint32)
        if self.model.n_rules:
            self._check(self._lib.sim_read_t_first(self._h, self.model.n_rules, _ptr(out)))
        return out[: self.model.n_rules]

    def load_t_first(self, t_first):
        a = np.ascontiguousarray(t_first, dtype=np.uint32)
        self._check(self._lib.sim_load_t_first(self._h, len(a), _ptr(a)))

    def debug_move_only(self):
        self._check(self._lib.sim_debug_move_only(self._h))

    def launch_count(self):
        return int(self._lib.sim_launch_count(self._h))

    def profile_enable(self, on=True):
        self._check(self._lib.sim_profile_enable(self._h, int(on)))

    def kernel_times(self):
        ms = np.zeros(N_KERNELS, dtype=np.float32)
        n = np.zeros(N_KERNELS, dtype=np.uint32)
        self._check(self._lib.sim_kernel_times(self._h, _ptr(ms), _ptr(n)))
        return {self._lib.sim_kernel_name(k).decode(): (float(ms[k]), int(n[k])) for k in range(N_KERNELS)}

    def monitor_eval(self, monitors, with_states=True):
        """monitors: dicts {replica, species (1..4 ids), threshold, first_row, n_rows}; sim_monitor_eval."""
        n = len(monitors)
        mons = (_Monitor * max(n, 1))()
        for i, m in enumerate(monitors):
            mons[i].replica, mons[i].n_species = m["replica"], len(m["species"])
            for k, sp in enumerate(m["species"][:4]):
                mons[i].species[k] = sp
            mons[i].threshold, mons[i].first_row, mons[i].n_rows = m["threshold"], m["first_row"], m["n_rows"]
        res = (_MonitorResult * max(n, 1))()
        stride = max([m["n_rows"] for m in monitors] + [1])
        states = np.zeros((max(n, 1), stride), dtype=np.uint8)
        self._check(self._lib.sim_monitor_eval(self._h, mons, n, res, _ptr(states) if with_states else None, stride))
        out = []
        for i, m in enumerate(monitors):
            d = {k: int(getattr(res[i], k)) for k, _ in _MonitorResult._fields_}
            if with_states:
                d["states"] = states[i, :m["n_rows"]].copy()
            out.append(d)
        return out


    def render(self, replica=0, axis=2, u0=0, v0=0, eu=None, ev=None, width=256, height=256, gain=255, palette=None):
        """RGBA8 picture of the live agents of one replica, coloured by compartment; sim_render."""
        ext = [e for a, e in enumerate(self.model.extent) if a != axis]
        if axis != 0 and self.model.n_replicas > 1:
            ext[0] = min(ext[0], 1 << self.model.stride_shift)
        v = _View()
        v.replica, v.axis, v.u0, v.v0 = replica, axis, u0, v0
        v.eu, v.ev = (ext[0] if eu is None else eu), (ext[1] if ev is None else ev)
        v.width, v.height, v.gain = width, height, gain
        palette = palette or [(255, 165, 0), (255, 255, 0)]     # cytoplasm orange, nucleus yellow
        for c in range(min(8, len(palette))):
            for k in range(3):
                v.palette[c][k] = palette[c][k]
        img = np.zeros((height, width, 4), dtype=np.uint8)
        self._check(self._lib.sim_render(self._h, C.byref(v), _ptr(img)))
        return img


def debug_philox(ctr, key):
    """Device Philox4x32-10 on (n,4) counters and (n,2) keys (test hook)."""
    import torch

    L = load_library()
    c = torch.from_numpy(np.ascontiguousarray(ctr, dtype=np.uint32).view(np.int32)).cuda()
    k = torch.from_numpy(np.ascontiguousarray(key, dtype=np.uint32).view(np.int32)).cuda()
    out = torch.empty_like(c)
    st = torch.cuda.current_stream().cuda_stream
    code = L.sim_debug_philox(C.c_void_p(c.data_ptr()), C.c_void_p(k.data_ptr()), C.c_void_p(out.data_ptr()),
                              c.shape[0], C.c_void_p(st))
    if code != 0:
        raise SimError(code)
    torch.cuda.synchronize()
    return out.cpu().numpy().view(np.uint32)
