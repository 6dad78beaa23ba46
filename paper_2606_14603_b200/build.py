"""Builds paper_2606_14603_b200/libmolsim.so with nvcc for sm_100a (in-tree, no JIT cache)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
# MOLSIM_CHECKS=1: the checked build (device-side bound checks on every data-derived index, csrc/device_types.cuh)
CHECKED = os.environ.get("MOLSIM_CHECKS") == "1"
LIB = os.path.join(HERE, "libmolsim_checked.so" if CHECKED else "libmolsim.so")
SRC = os.path.join(HERE, "csrc", "molsim.cu")
DEPS = [SRC, os.path.join(HERE, "csrc", "kernels.cuh"), os.path.join(HERE, "csrc", "device_types.cuh"),
        os.path.join(HERE, "csrc", "readout.cuh"), os.path.join(HERE, "csrc", "ptx_sm100.cuh"),
        os.path.join(os.path.dirname(HERE), "include", "molsim.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-shared", "-Xcompiler", "-fPIC", "-o", LIB, SRC]
    if CHECKED:
        cmd.insert(1, "-DMOLSIM_CHECKS=1")
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
