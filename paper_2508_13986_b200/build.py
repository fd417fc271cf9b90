"""Build libgbees.so (hand-written CUDA for sm_100a) in-tree with nvcc."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgbees.so")
SOURCES = [os.path.join(CSRC, "gbees_api.cu"), os.path.join(CSRC, "gbees_ht.cu"), os.path.join(CSRC, "gbees_noalloc.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("gbees_common.cuh", "gbees_prims.cuh", "gbees_brick.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "gbees.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--extended-lambda", "-shared", "-Xcompiler", "-fPIC"]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(
            os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS if os.path.exists(d)):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    dev = ["-DGBEES_DEV_PAIRS"] if os.environ.get("GBEES_DEV_PAIRS") else []   # development only: a subset of (n, dynamics)
    cmd = [nvcc, "--threads", "0"] + NVCC_FLAGS + dev + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
