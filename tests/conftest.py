import ctypes
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long statistical run")


@pytest.fixture(scope="session")
def torch_philox():
    """PyTorch's own CPU Philox4x32-10 (library routine) behind a C function; see helpers/."""
    import torch

    inc = os.path.join(os.path.dirname(torch.__file__), "include")
    src = os.path.join(ROOT, "tests", "helpers", "torch_philox.cpp")
    out = os.path.join(ROOT, "tests", "helpers", "libtorch_philox.so")
    if not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.run(["g++", "-O1", "-std=c++17", "-shared", "-fPIC", "-I" + inc, "-o", out, src], check=True)
    lib = ctypes.CDLL(out)
    lib.torch_philox4x32_10.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64]
    lib.torch_philox4x32_10.restype = None

    def f(ctr, key):
        ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
        key = np.ascontiguousarray(np.broadcast_to(np.asarray(key, dtype=np.uint32).reshape(-1, 2),
                                                   (ctr.shape[0], 2)))
        out_ = np.zeros_like(ctr)
        lib.torch_philox4x32_10(ctr.ctypes.data, key.ctypes.data, out_.ctypes.data, ctr.shape[0])
        return out_

    return f
