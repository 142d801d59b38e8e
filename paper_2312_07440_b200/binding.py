"""Thin ctypes binding of include/rwgt.h — argument marshalling only; every step of the hot path
runs in the CUDA kernels of librwgt.so.  Fails loudly when the library is missing or cannot load:
there is no CPU fallback."""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librwgt.so")

RWGT_FP64, RWGT_FP32, RWGT_MIXED = 0, 1, 2
PRECISIONS = {"fp64": RWGT_FP64, "fp32": RWGT_FP32, "mixed": RWGT_MIXED}

RWGT_MAX_SETS = 16
RWGT_MAX_PROCESSES = 4
EXPORTS = ("rwgt_create", "rwgt_create_multi", "rwgt_n_sets", "rwgt_run_multi", "rwgt_run_multi_host", "rwgt_set_precision", "rwgt_n_external", "rwgt_flops_per_event", "rwgt_run",
           "rwgt_run_host", "rwgt_destroy", "rwgt_last_error", "rwgt_colour_matrix", "rwgt_tensor_flops_per_event", "rwgt_sum_weights", "rwgt_run_file",
           "rwgt_create_multiprocess", "rwgt_n_processes", "rwgt_run_multiprocess", "rwgt_sum_weights_static", "rwgt_build_id")
RWGT_STATIC_SUM_MAX_ROWS = 17


class rwgt_params(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("alpha_em", "alpha_s", "mZ", "GammaZ", "sin2_thetaW", "mt",
                                          "Gamma_t", "ggg_scale", "gggg_scale")]


_lib = None


def lib():
    """Load librwgt.so (built by `python -m paper_2312_07440_b200.build` / __graft_entry__.build())."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not built: run `python paper_2312_07440_b200/build.py` "
                               "(the reweighting path has no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, dp = C.c_void_p, C.c_void_p
        L.rwgt_create.argtypes = [C.c_char_p, C.POINTER(rwgt_params), C.POINTER(rwgt_params)]
        L.rwgt_create.restype = vp
        L.rwgt_create_multi.argtypes = [C.c_char_p, C.POINTER(rwgt_params), C.POINTER(rwgt_params), C.c_int]
        L.rwgt_create_multi.restype = vp
        L.rwgt_n_sets.argtypes = [vp]
        L.rwgt_run_multi.argtypes = [vp, dp, dp, dp, dp, dp, C.c_longlong, vp]
        L.rwgt_run_multi_host.argtypes = [vp, dp, dp, dp, dp, dp, C.c_longlong, vp]
        L.rwgt_set_precision.argtypes = [vp, C.c_int]
        L.rwgt_n_external.argtypes = [vp]
        L.rwgt_flops_per_event.argtypes = [vp]
        L.rwgt_flops_per_event.restype = C.c_double
        L.rwgt_tensor_flops_per_event.argtypes = [vp]
        L.rwgt_tensor_flops_per_event.restype = C.c_double
        L.rwgt_run.argtypes = [vp, dp, dp, dp, dp, dp, C.c_longlong, vp]
        L.rwgt_run_host.argtypes = [vp, dp, dp, dp, dp, dp, C.c_longlong, vp]
        L.rwgt_destroy.argtypes = [vp]
        L.rwgt_last_error.restype = C.c_char_p
        L.rwgt_build_id.restype = C.c_char_p
        L.rwgt_colour_matrix.argtypes = [C.c_int, dp]
        L.rwgt_create_multiprocess.argtypes = [C.c_char_p, C.POINTER(rwgt_params), C.POINTER(rwgt_params), C.c_int]
        L.rwgt_create_multiprocess.restype = vp
        L.rwgt_n_processes.argtypes = [vp]
        L.rwgt_run_multiprocess.argtypes = [vp, dp, dp, dp, dp, dp, dp, C.c_longlong, vp]
        L.rwgt_sum_weights.argtypes = [vp, dp, C.c_int, C.c_longlong, dp, vp]
        L.rwgt_sum_weights_static.argtypes = [dp, C.c_int, C.c_longlong, dp, vp]
        L.rwgt_run_file.argtypes = [vp, C.c_char_p, C.c_char_p, C.c_longlong, C.c_longlong, vp]
        _lib = L
    return _lib


def _params(p) -> rwgt_params:
    if isinstance(p, rwgt_params):
        return p
    return rwgt_params(*[float(x) for x in p])


def rwgt_last_error() -> str:
    return lib().rwgt_last_error().decode()


def rwgt_create(process: str, params_old, params_new):
    po, pn = _params(params_old), _params(params_new)
    h = lib().rwgt_create(process.encode(), C.byref(po), C.byref(pn))
    if not h:
        raise RuntimeError(rwgt_last_error())
    return h


def rwgt_create_multi(process: str, params_old, params_new_list):
    """K new parameter sets for the same events (PAPER.md:87 step 7)."""
    po = _params(params_old)
    arr = (rwgt_params * len(params_new_list))(*[_params(p) for p in params_new_list])
    h = lib().rwgt_create_multi(process.encode(), C.byref(po), arr, len(params_new_list))
    if not h:
        raise RuntimeError(rwgt_last_error())
    return h


def rwgt_create_multiprocess(processes: str, params_old, params_new_list):
    """LO multiprocess: comma-separated process names sharing n_ext, K new parameter sets."""
    po = _params(params_old)
    arr = (rwgt_params * len(params_new_list))(*[_params(p) for p in params_new_list])
    h = lib().rwgt_create_multiprocess(processes.encode(), C.byref(po), arr, len(params_new_list))
    if not h:
        raise RuntimeError(rwgt_last_error())
    return h


def rwgt_n_processes(h) -> int:
    return lib().rwgt_n_processes(h)


def rwgt_run_multiprocess(h, momenta_ptr: int, weights_ptr: int, process_id: np.ndarray, out_me_old_ptr: int, out_me_new_ptr: int,
                          out_w_new_ptr: int, n_events: int, stream: int = 0) -> None:
    """Device pointers for the event buffers; process_id is a HOST int32 array [n_events]."""
    assert process_id.dtype == np.int32 and process_id.flags.c_contiguous and process_id.shape == (int(n_events),)
    rc = lib().rwgt_run_multiprocess(h, momenta_ptr, weights_ptr, process_id.ctypes.data, out_me_old_ptr, out_me_new_ptr, out_w_new_ptr,
                                     int(n_events), stream or None)
    if rc != 0:
        raise RuntimeError(f"rwgt_run_multiprocess rc={rc}: {rwgt_last_error()}")


def rwgt_n_sets(h) -> int:
    return lib().rwgt_n_sets(h)


def rwgt_build_id() -> str:
    """SHA-256 prefix of the sources librwgt.so was built from (build.py source_id)."""
    return lib().rwgt_build_id().decode()


def rwgt_set_precision(h, mode) -> None:
    mode = PRECISIONS.get(mode, mode)
    if lib().rwgt_set_precision(h, int(mode)) != 0:
        raise RuntimeError(rwgt_last_error())


def rwgt_n_external(h) -> int:
    return lib().rwgt_n_external(h)


def rwgt_flops_per_event(h) -> float:
    return lib().rwgt_flops_per_event(h)


def rwgt_tensor_flops_per_event(h) -> float:
    return lib().rwgt_tensor_flops_per_event(h)


def rwgt_run(h, momenta_ptr: int, weights_ptr: int, out_me_old_ptr: int, out_me_new_ptr: int,
             out_w_new_ptr: int, n_events: int, stream: int = 0) -> None:
    """Device pointers (ints, e.g. torch.Tensor.data_ptr()) and a cudaStream_t handle."""
    rc = lib().rwgt_run(h, momenta_ptr, weights_ptr, out_me_old_ptr, out_me_new_ptr, out_w_new_ptr,
                        int(n_events), stream or None)
    if rc != 0:
        raise RuntimeError(f"rwgt_run rc={rc}: {rwgt_last_error()}")


def rwgt_run_multi(h, momenta_ptr: int, weights_ptr: int, out_me_old_ptr: int, out_me_new_ptr: int,
                   out_w_new_ptr: int, n_events: int, stream: int = 0) -> None:
    """As rwgt_run for K = rwgt_n_sets(h) new sets: out_me_new / out_w_new are device [K][n_events]."""
    rc = lib().rwgt_run_multi(h, momenta_ptr, weights_ptr, out_me_old_ptr, out_me_new_ptr, out_w_new_ptr,
                              int(n_events), stream or None)
    if rc != 0:
        raise RuntimeError(f"rwgt_run_multi rc={rc}: {rwgt_last_error()}")


def rwgt_run_multi_host(h, momenta: np.ndarray, weights: np.ndarray, out_me_old: np.ndarray,
                        out_me_new: np.ndarray, out_w_new: np.ndarray, stream: int = 0) -> None:
    """Host numpy buffers; out_me_new / out_w_new have shape (K, n)."""
    n = weights.shape[0]
    for a in (momenta, weights, out_me_old, out_me_new, out_w_new):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    assert out_me_new.shape == (rwgt_n_sets(h), n) and out_w_new.shape == (rwgt_n_sets(h), n)
    rc = lib().rwgt_run_multi_host(h, momenta.ctypes.data, weights.ctypes.data, out_me_old.ctypes.data,
                                   out_me_new.ctypes.data, out_w_new.ctypes.data, int(n), stream or None)
    if rc != 0:
        raise RuntimeError(f"rwgt_run_multi_host rc={rc}: {rwgt_last_error()}")


def rwgt_run_host(h, momenta: np.ndarray, weights: np.ndarray, out_me_old: np.ndarray,
                  out_me_new: np.ndarray, out_w_new: np.ndarray, stream: int = 0) -> None:
    """Host numpy buffers (float64, C-contiguous); copies in/out inside the call."""
    n = weights.shape[0]
    for a in (momenta, weights, out_me_old, out_me_new, out_w_new):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    rc = lib().rwgt_run_host(h, momenta.ctypes.data, weights.ctypes.data, out_me_old.ctypes.data,
                             out_me_new.ctypes.data, out_w_new.ctypes.data, int(n), stream or None)
    if rc != 0:
        raise RuntimeError(f"rwgt_run_host rc={rc}: {rwgt_last_error()}")


def rwgt_sum_weights(h, w_ptr: int, n_rows: int, n_events: int, out_sums_ptr: int, stream: int = 0) -> None:
    """eq. 2: device pointers; w is [n_rows][n_events], out_sums [n_rows]."""
    rc = lib().rwgt_sum_weights(h, w_ptr, int(n_rows), int(n_events), out_sums_ptr, stream or None)
    if rc != 0:
        raise RuntimeError(f"rwgt_sum_weights rc={rc}: {rwgt_last_error()}")


def rwgt_sum_weights_static(w_ptr: int, n_rows: int, n_events: int, out_sums_ptr: int, stream: int = 0) -> None:
    """eq. 2 for a caller that may not allocate device memory (all of it belongs to the host program's own arena,
    or a cudaMalloc's device-wide wait is not affordable): no handle, no allocation; the reduction's scratch is a fixed 9 KB array
    inside librwgt.so.  Device pointers on the current device; w is [n_rows][n_events], out_sums [n_rows]; n_rows <= 17
    (RWGT_STATIC_SUM_MAX_ROWS), more raises.  All calls on a device share that array: keep them stream-ordered.  Make the first
    call on a device at set-up, outside any stream capture (it looks up the array's device address)."""
    rc = lib().rwgt_sum_weights_static(w_ptr, int(n_rows), int(n_events), out_sums_ptr, stream or None)
    if rc != 0:
        raise RuntimeError(f"rwgt_sum_weights_static rc={rc}: {rwgt_last_error()}")


def rwgt_run_file(h, in_path: str, out_path: str, first_event: int = 0, n_events: int = -1, stream: int = 0) -> None:
    """PAPER.md:87 steps 2-8 on a binary SoA event file: read -> H2D -> kernel -> D2H -> write (pipelined in the library)."""
    rc = lib().rwgt_run_file(h, os.fsencode(in_path), os.fsencode(out_path), int(first_event), int(n_events), stream or None)
    if rc != 0:
        raise RuntimeError(f"rwgt_run_file rc={rc}: {rwgt_last_error()}")


# ---- event / result files (layout: include/rwgt.h rwgt_event_file_header / rwgt_result_file_header); byte shuffling only ----
_EVT_HDR = np.dtype([("magic", "S8"), ("version", "<u4"), ("n_ext", "<u4"), ("n_events", "<u8"), ("process", "S32"), ("reserved", "<u8")])
_RES_HDR = np.dtype([("magic", "S8"), ("version", "<u4"), ("n_sets", "<u4"), ("n_events", "<u8"), ("process", "S32"), ("first_event", "<u8")])
assert _EVT_HDR.itemsize == 64 and _RES_HDR.itemsize == 64


def write_event_file(path: str, process: str, momenta: np.ndarray, weights: np.ndarray) -> None:
    """momenta[n_ext,4,n] (E,px,py,pz), weights[n], float64: the stand-in for an LHE event file (PAPER.md:87 step 2)."""
    n_ext, four, n = momenta.shape
    assert four == 4 and weights.shape == (n,) and momenta.dtype == np.float64 and weights.dtype == np.float64
    hd = np.zeros(1, dtype=_EVT_HDR)
    hd["magic"], hd["version"], hd["n_ext"], hd["n_events"], hd["process"] = b"RWGTEVT1", 1, n_ext, n, process.encode()
    with open(path, "wb") as f:
        f.write(hd.tobytes())
        f.write(np.ascontiguousarray(momenta).tobytes())
        f.write(np.ascontiguousarray(weights).tobytes())


def read_event_file(path: str):
    """-> (process, momenta[n_ext,4,n], weights[n])."""
    with open(path, "rb") as f:
        hd = np.frombuffer(f.read(64), dtype=_EVT_HDR)[0]
        if hd["magic"] != b"RWGTEVT1" or hd["version"] != 1:
            raise ValueError(f"{path}: not an event file")
        n_ext, n = int(hd["n_ext"]), int(hd["n_events"])
        m = np.frombuffer(f.read(n_ext * 4 * n * 8), dtype="<f8").reshape(n_ext, 4, n)
        w = np.frombuffer(f.read(n * 8), dtype="<f8")
    return hd["process"].decode(), m, w


def event_file_n_events(path: str) -> int:
    with open(path, "rb") as f:
        hd = np.frombuffer(f.read(64), dtype=_EVT_HDR)[0]
    if hd["magic"] != b"RWGTEVT1":
        raise ValueError(f"{path}: not an event file")
    return int(hd["n_events"])


def event_file_process(path: str) -> str:
    with open(path, "rb") as f:
        hd = np.frombuffer(f.read(64), dtype=_EVT_HDR)[0]
    return hd["process"].decode()


def read_result_file(path: str) -> dict:
    """-> dict(process, first_event, me_old[n], me_new[K,n], w_new[K,n], sum_w_old, sum_w_new[K])."""
    with open(path, "rb") as f:
        hd = np.frombuffer(f.read(64), dtype=_RES_HDR)[0]
        if hd["magic"] != b"RWGTRES1" or hd["version"] != 1:
            raise ValueError(f"{path}: not a result file")
        K, n = int(hd["n_sets"]), int(hd["n_events"])
        body = np.frombuffer(f.read(((1 + 2 * K) * n + 1 + K) * 8), dtype="<f8")
    rows = body[: (1 + 2 * K) * n].reshape(1 + 2 * K, n)
    sums = body[(1 + 2 * K) * n:]
    return {"process": hd["process"].decode(), "first_event": int(hd["first_event"]), "me_old": rows[0], "me_new": rows[1:1 + K],
            "w_new": rows[1 + K:], "sum_w_old": float(sums[0]), "sum_w_new": sums[1:].copy()}


def rwgt_destroy(h) -> None:
    lib().rwgt_destroy(h)


def rwgt_colour_matrix(n_gluons: int) -> np.ndarray:
    f = math.factorial(n_gluons)
    out = np.empty((f, f), dtype=np.float64)
    if lib().rwgt_colour_matrix(n_gluons, out.ctypes.data) != f:
        raise RuntimeError("rwgt_colour_matrix: bad n_gluons")
    return out


class Reweighter:
    """Convenience wrapper: one handle, torch device tensors in, torch device tensors out."""

    def __init__(self, process: str, params_old, params_new, precision="fp64"):
        """params_new: one parameter set, or a list of K sets (then run() returns 1 + 2K rows:
        |M|^2, K rows |M'_k|^2, K rows W'_k)."""
        multi = isinstance(params_new, list)
        self.multiprocess = "," in process            # "gg_ttxg,qqx_ttxg": run() then needs process_id
        if self.multiprocess:
            self.h = rwgt_create_multiprocess(process, params_old, params_new if multi else [params_new])
        else:
            self.h = rwgt_create_multi(process, params_old, params_new) if multi else rwgt_create(process, params_old, params_new)
        self.k = rwgt_n_sets(self.h)
        self.process = process
        self.n_ext = rwgt_n_external(self.h)
        rwgt_set_precision(self.h, precision)

    def flops_per_event(self) -> float:
        return rwgt_flops_per_event(self.h)

    def tensor_flops_per_event(self) -> float:
        return rwgt_tensor_flops_per_event(self.h)

    def run(self, momenta, weights, out=None, process_id=None):
        import torch
        n = weights.shape[0]
        assert momenta.is_cuda and momenta.dtype == torch.float64 and momenta.is_contiguous()
        assert momenta.shape == (self.n_ext, 4, n)
        assert weights.is_cuda and weights.dtype == torch.float64 and weights.is_contiguous() and weights.device == momenta.device
        k = self.k
        if out is None:
            out = torch.empty((1 + 2 * k, n), dtype=torch.float64, device=momenta.device)
        assert out.is_cuda and out.dtype == torch.float64 and out.device == momenta.device
        assert out.shape == (1 + 2 * k, n) and out.is_contiguous()
        st = torch.cuda.current_stream(momenta.device).cuda_stream
        if self.multiprocess:
            rwgt_run_multiprocess(self.h, momenta.data_ptr(), weights.data_ptr(), np.ascontiguousarray(process_id, dtype=np.int32),
                                  out[0].data_ptr(), out[1].data_ptr(), out[1 + k].data_ptr(), n, st)
            return out
        rwgt_run_multi(self.h, momenta.data_ptr(), weights.data_ptr(), out[0].data_ptr(), out[1].data_ptr(),
                       out[1 + k].data_ptr(), n, st)
        return out

    def cross_sections(self, w_rows):
        """eq. 2: sum of every row of a device tensor [rows, n] (e.g. run()[1 + K:], the K reweighted sets)."""
        import torch
        assert w_rows.is_cuda and w_rows.dtype == torch.float64 and w_rows.is_contiguous() and w_rows.dim() == 2
        out = torch.empty(w_rows.shape[0], dtype=torch.float64, device=w_rows.device)
        rwgt_sum_weights(self.h, w_rows.data_ptr(), w_rows.shape[0], w_rows.shape[1], out.data_ptr(), torch.cuda.current_stream(w_rows.device).cuda_stream)
        return out

    def close(self):
        if self.h:
            rwgt_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
