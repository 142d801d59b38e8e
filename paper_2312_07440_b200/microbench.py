"""ctypes binding of include/rwgt_microbench.h (librwgt_microbench.so): FMA-chain peak measurements for bench.py's roofline.
A measurement aid, separate from the reweighting library."""
import ctypes as C
import os

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "librwgt_microbench.so")
EXPORTS = ("rwgt_microbench_peak",)
_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not built: run `python paper_2312_07440_b200/build.py`")
        _lib = C.CDLL(LIB_PATH)
        _lib.rwgt_microbench_peak.argtypes = [C.c_int, C.POINTER(C.c_double)]
    return _lib


def rwgt_microbench_peak(kind: int) -> float:
    """TFLOP/s of microbenchmark `kind` (see include/rwgt_microbench.h) on the current CUDA device."""
    out = C.c_double()
    if lib().rwgt_microbench_peak(int(kind), C.byref(out)) != 0:
        raise RuntimeError("rwgt_microbench_peak failed")
    return out.value
