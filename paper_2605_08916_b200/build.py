"""Builds paper_2605_08916_b200/libdr.so (the C-ABI library of include/dr.h) with nvcc for sm_100a, in-tree."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdr.so")
SOURCES = ["dr_api.cu", "dr_bvh.cpp"]
DEPS = SOURCES + ["dr_kernels.cuh", "dr_eval.cuh", "dr_wave.cuh", "dr_traverse.cuh", "dr_path.cuh", "dr_rng.cuh", "dr_types.h", "../../include/dr.h"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
               "-Xcompiler", "-fPIC", "-o", LIB]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        cmd += os.environ.get("DR_NVCC_FLAGS", "").split()   # e.g. -DDR_TRACE_BLOCK=640 for a tuning sweep
        cmd += [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
