"""TEST INFRASTRUCTURE: builds tests/simt/_build/libmolsim_simt[_san].so, the product's CUDA sources compiled for the
host against the SIMT emulation of simt_shim.h.  The sources are taken from paper_2606_14603_b200/csrc/ as they are,
apart from three mechanical rewrites g++ needs:
  * `kernel<<<grid, block, smem, stream>>>(` -> `simt::cfg(grid, block, smem, stream).call(kernel)(`
  * `extern __shared__ [__align__(n)] T name[];` -> `T* name = (T*)simt::dyn_smem();`
  * ptx_sm100.cuh (inline PTX) is replaced by ptx_sm100_emu.cuh (the same helpers with the PTX ISA's semantics)
Nothing under paper_2606_14603_b200/ imports, builds or loads this; it is not a CPU fallback (see simt_shim.h)."""
import os
import re
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_2606_14603_b200", "csrc")
OUT = os.path.join(HERE, "_build")

LAUNCH = re.compile(r"([A-Za-z_][\w:>\-]*(?:<[\w, ]*>)?)<<<(.*?)>>>\(", re.S)
DYN_SMEM = re.compile(r"extern\s+__shared__\s+(?:__align__\(\d+\)\s+)?(\w+)\s+(\w+)\[\];")


def transform(text: str) -> str:
    text = LAUNCH.sub(lambda m: f"simt::cfg({m.group(2)}).call({m.group(1)})(", text)
    text = DYN_SMEM.sub(lambda m: f"{m.group(1)}* {m.group(2)} = ({m.group(1)}*)simt::dyn_smem();", text)
    return text.replace('#include "../../include/molsim.h"', f'#include "{os.path.join(ROOT, "include", "molsim.h")}"')


def lib_path(sanitize: bool) -> str:
    return os.path.join(OUT, "libmolsim_simt_san.so" if sanitize else "libmolsim_simt.so")


def build(sanitize: bool = False, force: bool = False) -> str:
    lib = lib_path(sanitize)
    src_dir = os.path.join(OUT, "src")
    os.makedirs(src_dir, exist_ok=True)
    deps = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh"))]
    deps += [os.path.join(HERE, f) for f in ("simt_shim.h", "simt_runtime.cpp", "ptx_sm100_emu.cuh", "build.py")]
    deps.append(os.path.join(ROOT, "include", "molsim.h"))
    if not force and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in deps):
        return lib
    n_launches = 0
    for name in sorted(os.listdir(CSRC)):
        if not name.endswith((".cu", ".cuh")):
            continue
        text = open(os.path.join(CSRC, name)).read()
        if name == "ptx_sm100.cuh":
            text = open(os.path.join(HERE, "ptx_sm100_emu.cuh")).read()
        else:
            n_launches += text.count("<<<")
            text = transform(text)
            assert "<<<" not in text and "asm volatile" not in text, f"{name}: a construct the rewrite does not know"
        with open(os.path.join(src_dir, name.replace(".cu", ".cpp") if name.endswith(".cu") else name), "w") as f:
            f.write(text)
    assert n_launches > 0
    with open(os.path.join(src_dir, "cuda_runtime.h"), "w") as f:
        f.write("// emulation build: simt_shim.h (force-included) stands in for the CUDA runtime\n")
    cmd = ["g++", "-std=c++17", "-g", "-fPIC", "-shared", "-DMOLSIM_CHECKS=1", "-include", os.path.join(HERE, "simt_shim.h"),
           "-I", src_dir, "-I", HERE, "-Wno-unknown-pragmas", "-Wno-attributes", "-o", lib,
           os.path.join(src_dir, "molsim.cpp"), os.path.join(HERE, "simt_runtime.cpp")]
    cmd[1:1] = (["-O1", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
                if sanitize else ["-O2"])
    subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    import sys
    print(build(sanitize="--san" in sys.argv, force=True))
