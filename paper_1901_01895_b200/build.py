"""Build libmmf_b200.so (the C-ABI CUDA library of include/mmf.h) in-tree with nvcc for sm_100a."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmmf_b200.so")
SOURCES = [os.path.join(CSRC, "mmf_api.cu"), os.path.join(CSRC, "probes.cu"), os.path.join(CSRC, "nl_static.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("fft_core.cuh", "fft_kernels.cuh", "nl_tma.cuh", "async_copy.cuh", "nl_simt.cuh", "nl_general.cuh", "nl_shard.cuh", "small_cluster.cuh", "tmem_exchange.cuh", "probes.cu")] + [
    os.path.join(os.path.dirname(HERE), "include", "mmf.h")]


def nvcc_path():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc_path(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-o", tmp] + SOURCES
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
