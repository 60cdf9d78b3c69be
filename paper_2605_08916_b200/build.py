"""Builds paper_2605_08916_b200/libdr.so (the C-ABI library of include/dr.h) with nvcc for sm_100a, in-tree."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdr.so")
SOURCES = ["dr_api.cu", "dr_bvh.cpp"]
DEPS = SOURCES + ["dr_kernels.cuh", "dr_eval.cuh", "dr_wave.cuh", "dr_grad.cuh", "dr_nee.cuh", "dr_traverse.cuh", "dr_path.cuh", "dr_rng.cuh",
                  "dr_types.h", "../../include/dr.h"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
# -fmad=false: no implicit contraction of a * b + c; the kernels say fmaf() where they want one (traversal), and the path
# arithmetic rounds like a plain fp32 evaluation of the formulas of DESIGN.md Q4-Q8 (csrc/dr_path.cuh, Q15)
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-fmad=false", "-shared", "-Xcompiler", "-fPIC"]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = [NVCC] + FLAGS + ["-o", LIB]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        cmd += os.environ.get("DR_NVCC_FLAGS", "").split()   # e.g. -DDR_TRACE_BLOCK=640 for a tuning sweep
        cmd += [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True, cwd=CSRC)
    return LIB


def build_variant(name: str, flags: list) -> str:
    """A second library with extra compile flags (tests: e.g. the stalled-consumer build of k_wave); load it by pointing
    DR_LIB at the returned path before importing the package."""
    lib = os.path.join(HERE, f"libdr_{name}.so")
    if not os.path.exists(lib) or any(os.path.getmtime(os.path.join(CSRC, f)) > os.path.getmtime(lib) for f in DEPS):
        cmd = [NVCC] + FLAGS + ["-o", lib] + list(flags) + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True, cwd=CSRC)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
