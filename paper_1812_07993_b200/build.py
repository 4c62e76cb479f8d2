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


def build_operand_bench() -> str:
    """Compiles the stand-alone FP64 operand-pattern diagnostic (csrc/fp64_operand_bench.cu; profiles/r02_counters.md
    section 3) into build/fp64_operand_bench at the repository root.  Not part of the library."""
    out_dir = os.path.join(HERE, "..", "build")
    os.makedirs(out_dir, exist_ok=True)
    exe = os.path.join(out_dir, "fp64_operand_bench")
    subprocess.run([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                    os.path.join(HERE, "csrc", "fp64_operand_bench.cu"), "-o", exe], check=True)
    return os.path.abspath(exe)


if __name__ == "__main__":
    import sys
    if "--operand-bench" in sys.argv[1:]:
        print(build_operand_bench())
    else:
        print(build(force=True, verbose=True))
