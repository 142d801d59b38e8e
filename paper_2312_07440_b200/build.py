"""Build paper_2312_07440_b200/librwgt.so (the C-ABI library of include/rwgt.h) for sm_100a, in-tree."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librwgt.so")
LIB_EXP = os.path.join(HERE, "librwgt_exp.so")
SOURCES = [os.path.join(CSRC, "rwgt_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("rwgt_math.cuh", "kernels_small.cuh", "bg_engine.cuh", "photon_kernel.cuh", "microbench.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "rwgt.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "--fmad=true"]


def up_to_date() -> bool:
    return os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS)


def build(force: bool = False, verbose: bool = False, experiment: bool = False) -> str:
    """experiment=True builds librwgt_exp.so with -DRWGT_EXPERIMENT (the phase-removal switches of experiments.py)."""
    lib = LIB_EXP if experiment else LIB
    if not force and not experiment and up_to_date():
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-DRWGT_EXPERIMENT"] if experiment else []) + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + SOURCES
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, experiment="--experiment" in sys.argv))
