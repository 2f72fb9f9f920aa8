"""Build libmmf_b200.so (the C-ABI CUDA library of include/mmf.h) and libmmf_probes.so (the measurement probes of
include/mmf_probes.h, used by `bench.py --probes` only) in-tree with nvcc for sm_100a.

Every translation unit is compiled to an object of its own (kept under paper_1901_01895_b200/build/, git-ignored) and
recompiled only when it or one of the files it includes is newer; the objects are then linked into their library."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libmmf_b200.so")
PROBES_LIB = os.path.join(HERE, "libmmf_probes.so")
HEADER = os.path.join(os.path.dirname(HERE), "include", "mmf.h")
PROBES_HEADER = os.path.join(os.path.dirname(HERE), "include", "mmf_probes.h")
CUH = [os.path.join(CSRC, f) for f in ("fft_core.cuh", "fft_kernels.cuh", "nl_tma.cuh", "async_copy.cuh", "nl_simt.cuh",
                                       "nl_general.cuh", "nl_shard.cuh", "small_cluster.cuh", "tmem_exchange.cuh")]
# translation unit -> the files it includes (besides itself)
UNITS = {"mmf_api.cu": CUH + [HEADER], "probes.cu": CUH + [HEADER, PROBES_HEADER], "nl_static.cu": [HEADER],
         "noise.cu": [HEADER]}
LIBS = {LIB: ["mmf_api.cu", "nl_static.cu", "noise.cu"], PROBES_LIB: ["probes.cu"]}
SOURCES = [os.path.join(CSRC, u) for u in UNITS]
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]


def nvcc_path():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale(target, deps):
    return not os.path.exists(target) or any(os.path.getmtime(target) < os.path.getmtime(d) for d in deps)


def build(force=False, verbose=False):
    me = os.path.abspath(__file__)
    os.makedirs(OBJ, exist_ok=True)
    objs, procs = [], []
    for unit, deps in UNITS.items():
        src = os.path.join(CSRC, unit)
        obj = os.path.join(OBJ, unit.replace(".cu", ".o"))
        objs.append(obj)
        if force or _stale(obj, [src, me] + deps):
            cmd = [nvcc_path()] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj + ".tmp"]
            procs.append((obj, cmd, subprocess.Popen(cmd)))      # the units compile side by side
    for obj, cmd, pr in procs:
        if pr.wait() != 0:
            raise subprocess.CalledProcessError(pr.returncode, cmd)
        os.replace(obj + ".tmp", obj)
    for lib, units in LIBS.items():
        mine = [os.path.join(OBJ, u.replace(".cu", ".o")) for u in units]
        if _stale(lib, mine):
            tmp = lib + ".tmp.%d" % os.getpid()
            subprocess.run([nvcc_path(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + mine,
                           check=True)
            os.replace(tmp, lib)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
