"""TEST INFRASTRUCTURE: drives the emulation build of the CUDA sources (tests/simt/build.py) through the same ctypes
calls the product binding makes.  `SimtSim` is `paper_2606_14603_b200.Sim` with two differences: the library is
libmolsim_simt[_san].so and the "device" workspace is a garbage-filled host block from `simt_alloc`.  Tests only."""
import ctypes as C
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for p in (ROOT, HERE):
    if p not in sys.path:
        sys.path.insert(0, p)

import build as simt_build  # noqa: E402  (tests/simt/build.py)
from paper_2606_14603_b200 import binding  # noqa: E402

_libs = {}


def load(sanitize=False):
    if sanitize not in _libs:
        L = binding.declare_signatures(C.CDLL(simt_build.build(sanitize=sanitize)))
        L.simt_alloc.argtypes = [C.c_size_t]
        L.simt_alloc.restype = C.c_void_p
        L.simt_free.argtypes = [C.c_void_p]
        L.simt_free.restype = None
        L.simt_switches.restype = C.c_uint64
        L.simt_launches.restype = C.c_uint64
        _libs[sanitize] = L
    return _libs[sanitize]


class SimtSim(binding.Sim):
    def __init__(self, model, cell_size=None, seed=None, sanitize=False):
        self._lib = load(sanitize)
        self.model = model
        cfg, keep = binding.marshal_config(model, cell_size, seed)
        nbytes = self._lib.sim_workspace_bytes(C.byref(cfg))
        if nbytes == 0:
            why = self._lib.sim_check_config(C.byref(cfg))
            raise SimtError(binding.E_INVAL, self._lib, f"(sim_workspace_bytes: {why.decode() if why else 'cell grid too large'})")
        self._ws = self._lib.simt_alloc(nbytes)          # exactly the bytes asked for: one byte further is a red zone
        assert self._ws and self._ws % 256 == 0
        h = C.c_void_p()
        self._check(self._lib.sim_create(C.byref(cfg), C.c_void_p(self._ws), nbytes, None, C.byref(h)))
        self._h = h
        self.workspace_bytes = nbytes

    def _check(self, code):
        if code != 0:
            raise SimtError(code, self._lib)

    def close(self):
        super().close()
        if getattr(self, "_ws", None):
            self._lib.simt_free(self._ws)
            self._ws = None


class SimtError(binding.SimError):
    def __init__(self, code, lib, detail=""):
        RuntimeError.__init__(self, f"molsim (emulation) error {code}: {lib.sim_strerror(code).decode()} {detail}")
        self.code = code


class Emu:
    """Stands where the GPU test modules expect the package: `.Sim`, `.SimError`."""
    SimError = binding.SimError

    def __init__(self, sanitize=False):
        self.sanitize = sanitize

    def Sim(self, model, cell_size=None, seed=None, stream=None):
        return SimtSim(model, cell_size=cell_size, seed=seed, sanitize=self.sanitize)
