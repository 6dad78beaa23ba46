"""TEST INFRASTRUCTURE: builds tests/simt/_build/libmolsim_simt[_san].so, the product's CUDA sources compiled for the
host against the SIMT emulation of simt_shim.h.  The sources are taken from paper_2606_14603_b200/csrc/ as they are,
apart from three mechanical rewrites g++ needs:
  * `kernel<<<grid, block, smem, stream>>>(` -> `simt::cfg(grid, block, smem, stream).call(kernel)(`
  * `extern __shared__ [__align__(n)] T name[];` -> `T* name = (T*)simt::dyn_smem();`
  * ptx_sm100.cuh (inline PTX) is replaced by ptx_sm100_emu.cuh (the same helpers with the PTX ISA's semantics)
The ThreadSanitizer build (mode "tsan") makes four more (RACY_BY_DESIGN), for the races the kernels have BY DESIGN — the
plain `prop[]` stores of K4 (K4b checks them against the 64-bit key), K5's live read of `t_first` (equivalent to reading
it as of the start of the step) and the same-value stores with which K6 and k_clear_ids clear shared bitmap / counter words — which become
relaxed atomic accesses there.
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


RACY_BY_DESIGN = [
    ("p.prop[i] = j; p.prop[j] = i;", "simt::relaxed_store(&p.prop[i], j); simt::relaxed_store(&p.prop[j], i);"),
    ("*((volatile uint32_t*)&p.scal->t_first[ch.rule])", "simt::relaxed_load(&p.scal->t_first[ch.rule])"),
    # K6's epilogue clears the birth bitmap / counter words of every firing parent: parents that share a word store the same 0
    ("p.bits[pid >> 3] = 0u; p.birth_mid[pid >> kMidShift] = 0u; p.birth_top[pid >> p.top_shift] = 0u;",
     "simt::relaxed_store(&p.bits[pid >> 3], 0u); simt::relaxed_store(&p.birth_mid[pid >> kMidShift], 0u); "
     "simt::relaxed_store(&p.birth_top[pid >> p.top_shift], 0u);"),
    # ... and so does k_clear_ids (sim_load_agents) for ids that share a bitmap word
    ("if (id < p.id_capacity) p.bits[id >> 3] = 0u;", "if (id < p.id_capacity) simt::relaxed_store(&p.bits[id >> 3], 0u);"),
]


def lib_path(sanitize) -> str:
    return os.path.join(OUT, {False: "libmolsim_simt.so", True: "libmolsim_simt_san.so", "tsan": "libmolsim_simt_tsan.so"}[sanitize])


def build(sanitize=False, force: bool = False) -> str:
    """sanitize: False (plain -O2), True (AddressSanitizer + UBSan) or "tsan" (ThreadSanitizer on the kernels)."""
    lib = lib_path(sanitize)
    src_dir = os.path.join(OUT, "src_tsan" if sanitize == "tsan" else "src")
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
            if sanitize == "tsan" and name == "kernels.cuh":
                for old, new in RACY_BY_DESIGN:
                    assert text.count(old) == 1, old
                    text = text.replace(old, new)
            assert "<<<" not in text and "asm volatile" not in text, f"{name}: a construct the rewrite does not know"
        with open(os.path.join(src_dir, name.replace(".cu", ".cpp") if name.endswith(".cu") else name), "w") as f:
            f.write(text)
    assert n_launches > 0
    with open(os.path.join(src_dir, "cuda_runtime.h"), "w") as f:
        f.write("// emulation build: simt_shim.h (force-included) stands in for the CUDA runtime\n")
    common = ["g++", "-std=c++17", "-g", "-fPIC", "-DMOLSIM_CHECKS=1", "-include", os.path.join(HERE, "simt_shim.h"),
              "-I", src_dir, "-I", HERE, "-Wno-unknown-pragmas", "-Wno-attributes"]
    srcs = [os.path.join(src_dir, "molsim.cpp"), os.path.join(HERE, "simt_runtime.cpp")]
    tmp = f"{lib}.{os.getpid()}.tmp"
    if sanitize == "tsan":      # the kernels are instrumented, the scheduler is not (it only annotates: simt_runtime.cpp)
        objs = [os.path.join(OUT, f"tsan_molsim.{os.getpid()}.o"), os.path.join(OUT, f"tsan_runtime.{os.getpid()}.o")]
        subprocess.run(common + ["-O1", "-fsanitize=thread", "-DSIMT_TSAN=1", "-c", srcs[0], "-o", objs[0]], check=True)
        subprocess.run(common + ["-O2", "-DSIMT_TSAN=1", "-c", srcs[1], "-o", objs[1]], check=True)
        subprocess.run(["g++", "-shared", "-fsanitize=thread", "-o", tmp] + objs, check=True)
    else:
        opt = (["-O1", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
               if sanitize else ["-O2"])
        subprocess.run(common + opt + ["-shared", "-o", tmp] + srcs, check=True)
    os.replace(tmp, lib)          # a concurrent builder (pytest-xdist) never sees a half-written library
    return lib


if __name__ == "__main__":
    import sys
    print(build(sanitize="tsan" if "--tsan" in sys.argv else "--san" in sys.argv, force=True))
