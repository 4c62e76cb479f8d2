"""Compiles csrc/md_api.cu and csrc/md_noalloc.cu into paper_1812_07993_b200/libmd_b200.so for sm_100a (in-tree)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "csrc", "md_api.cu"), os.path.join(HERE, "csrc", "md_noalloc.cu")]
DEPS = SRCS + [os.path.join(HERE, "csrc", h) for h in ("md_kernels.cuh", "md_allpairs.cuh", "md_verlet.cuh")] + [
    os.path.join(HERE, "..", "include", "md.h")]
LIB = os.path.join(HERE, "libmd_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Xcompiler", "-fPIC", "-shared"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += os.environ.get("MD_NVCC_FLAGS", "").split()       # e.g. -DMD_DIAGNOSTICS (debug timers, standalone phase kernels)
    cmd += SRCS + ["-o", LIB]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
