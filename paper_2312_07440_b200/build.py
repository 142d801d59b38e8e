"""Build the in-tree CUDA libraries for sm_100a:
  librwgt.so             the C-ABI library of include/rwgt.h (the product)
  librwgt_microbench.so  include/rwgt_microbench.h, FMA-chain peak measurements used by bench.py only
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INC = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "librwgt.so")
LIB_MB = os.path.join(HERE, "librwgt_microbench.so")
TARGETS = {
    LIB: ([os.path.join(CSRC, "rwgt_api.cu")],
          [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cuh")] + [os.path.join(INC, "rwgt.h")]),
    LIB_MB: ([os.path.join(CSRC, "microbench.cu")], [os.path.join(INC, "rwgt_microbench.h")]),
}
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "--fmad=true"]


def source_id() -> str:
    """first 12 hex digits of the SHA-256 over librwgt.so's sources (what rwgt_build_id() returns)"""
    import hashlib
    h = hashlib.sha256()
    srcs, deps = TARGETS[LIB]
    for f in sorted(srcs + deps, key=os.path.basename):
        h.update(os.path.basename(f).encode() + b"\0" + open(f, "rb").read())
    return h.hexdigest()[:12]


def up_to_date(lib: str = LIB) -> bool:
    srcs, deps = TARGETS[lib]
    return os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in srcs + deps)


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    for lib, (srcs, _) in TARGETS.items():
        if not force and up_to_date(lib):
            continue
        ident = [f'-DRWGT_BUILD_ID="{source_id()}"'] if lib == LIB else []
        subprocess.check_call([nvcc] + NVCC_FLAGS + ident + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + srcs)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
