"""TEST INFRASTRUCTURE: does the emulation notice a synchronisation bug?  Each mutant is the emulation build of the CUDA
sources with ONE synchronisation removed from k_pairs / k_uni_hist / k_resolve (applied to the rewritten copy under
_build/, never to the product); `python mutants.py NAME SEED` builds it, runs a few parity cases against the oracle under
scheduler seed SEED (0 = the plain round-robin schedule) and exits 0 only if every case still matches, i.e. if the
mutant SURVIVED.  tests/test_simt_kernels.py expects every one of them to be killed (mismatch, bound check, deadlock
report or crash)."""
import ctypes as C
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path[:0] = [os.path.dirname(os.path.dirname(HERE)), os.path.dirname(HERE), HERE]

MUTANTS = {
    # the packed keys of the window are read by neighbouring lanes right after they are written
    "window_keys_without_syncwarp": ("      K[32u + lane] = pack_key(p, h.x, h.y, h.z);\n    }\n    __syncwarp();\n",
                                     "      K[32u + lane] = pack_key(p, h.x, h.y, h.z);\n    }\n"),
    # a stage of the ring is read before its bulk copy has landed (needs the late-landing copies of a seeded schedule)
    "tile_read_without_full_wait": ("    while (!mbar_try_wait(&S.full[stage], use & 1u)) {}\n",
                                    "    mbar_try_wait(&S.full[stage], use & 1u);\n"),
    # the hit counter is reset while other lanes may still be merging their hits
    "hit_reset_without_syncwarp": ("    __syncwarp();\n    if (lane == 0) S.nhit[warp] = 0;\n", "    if (lane == 0) S.nhit[warp] = 0;\n"),
    # K5's histogram part reads the tile's species before the unimolecular part has finished rewriting them
    "histogram_before_species_final": ("      __syncthreads();                      // the tile's species are final\n", "\n"),
    # K4b trusts prop[] (a racing plain store) without checking it against the 64-bit key
    "resolve_trusts_prop": ("      if (j >= n || (uint32_t)p.oth.r[j].w != idj) j = find_partner(&p, i, idj);\n", "\n"),
}


def main(name, seed):
    import build as sb

    sb.build()
    src, out = os.path.join(sb.OUT, "src"), os.path.join(sb.OUT, "mutant_" + name)
    os.makedirs(out, exist_ok=True)
    old, new = MUTANTS[name]
    for f in os.listdir(src):
        text = open(os.path.join(src, f)).read()
        if f == "kernels.cuh":
            assert text.count(old) == 1, f"{name}: the line to remove is not there (exactly once)"
            text = text.replace(old, new)
        open(os.path.join(out, f), "w").write(text)
    lib = os.path.join(out, "libmutant.so")
    subprocess.run(["g++", "-std=c++17", "-O1", "-fPIC", "-shared", "-DMOLSIM_CHECKS=1", "-include", os.path.join(HERE, "simt_shim.h"),
                    "-I", out, "-I", HERE, "-Wno-unknown-pragmas", "-Wno-attributes", "-o", lib,
                    os.path.join(out, "molsim.cpp"), os.path.join(HERE, "simt_runtime.cpp")], check=True)
    import harness
    from paper_2606_14603_b200 import binding

    L = binding.declare_signatures(C.CDLL(lib))
    L.simt_alloc.argtypes, L.simt_alloc.restype = [C.c_size_t], C.c_void_p
    L.simt_free.argtypes, L.simt_free.restype = [C.c_void_p], None
    harness._libs[False] = L
    os.environ["SIMT_SCHED_SEED"] = str(seed)
    import test_gpu_parity as gp
    import test_gpu_traces as gt

    emu = harness.Emu()
    gp.test_tiny_dense_cube_many_events(emu)
    gp.test_channel_kinds_and_priority(emu)
    gt.test_homodimer_parity(emu)
    print(f"MUTANT {name} SURVIVED seed {seed}")


if __name__ == "__main__":
    main(sys.argv[1], int(sys.argv[2]))
