"""Build libmps_b200.so (sm_100a only) in-tree with nvcc.

    python -m paper_2105_01677_b200.build [--force] [--verbose]

The library is plain CUDA runtime code behind a C ABI (include/mps_b200.h); it
links neither torch nor Python.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmps_b200.so")
SOURCES = ["mps_api.cu", "kernels_bin.cu", "kernels_sweep.cu", "kernels_ppe.cu", "no_alloc.cu"]
HEADERS = [os.path.join(CSRC, "mps_internal.h"),
           os.path.join(os.path.dirname(HERE), "include", "mps_b200.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fno-fast-math", "--fmad=true"]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    objs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(CSRC, src.replace(".cu", ".o"))
        if force or _stale(o, [s] + HEADERS):
            cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
            subprocess.check_call(cmd)
        objs.append(o)
    if force or _stale(LIB, objs):
        subprocess.check_call([NVCC, "-shared", "-o", LIB] + objs +
                              ["-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"])
    return LIB


def build_peaks() -> str:
    """The stand-alone ceilings micro-benchmark (microbench/peaks.cu, measurement tooling that is not
    part of libmps_b200.so; profiles/r01_ceilings_microbench.md) -> ./mps_peaks."""
    exe = os.path.join(HERE, "mps_peaks")
    src = os.path.join(HERE, "microbench", "peaks.cu")
    if _stale(exe, [src]):
        subprocess.check_call([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo",
                               "-std=c++17", "-o", exe, src])
    return exe


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    if "--peaks" in sys.argv:
        print(build_peaks())
