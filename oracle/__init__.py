"""ctypes front end of the CPU oracle (oracle/oracle.cpp).  TEST INFRASTRUCTURE ONLY:
imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
Nothing under paper_2312_07440_b200/ imports this package."""
from __future__ import annotations

import ctypes as C
import math
import numpy as np

from .build import build as _build

_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.orc_n_external.argtypes = [C.c_char_p]
        L.orc_me2.argtypes = [C.c_char_p, _dp, _dp, _dp]
        L.orc_reweight.argtypes = [C.c_char_p, _dp, _dp, _dp, _dp, _dp, _dp, _dp, C.c_long, C.c_int]
        L.orc_gamma.argtypes = [C.c_int, _dp]
        L.orc_spinor.argtypes = [C.c_int, _dp, C.c_double, C.c_int, _dp]
        L.orc_polvec.argtypes = [_dp, C.c_int, _dp]
        L.orc_colour_matrix.argtypes = [C.c_int, _dp]
        L.orc_fabc.argtypes = [_dp]
        L.orc_jamps.argtypes = [C.c_int, _dp, _dp, _ip, _dp, _dp]
        L.orc_me2_hel.argtypes = [C.c_int, _dp, _dp, _ip, C.c_int, _dp]
        L.orc_amp_epem.argtypes = [_dp, _dp, _ip, _dp]
        L.orc_amp_epem_ng.argtypes = [C.c_int, _dp, _dp, _ip, _dp, _dp]
        L.orc_cross_section.argtypes = [_dp, C.c_long]
        L.orc_cross_section.restype = C.c_double
        L.orc_me2_hel_qq.argtypes = [C.c_int, _dp, _dp, _ip, _dp, _dp]
        L.orc_denominator.argtypes = [C.c_int]
        L.orc_denominator.restype = C.c_double
        _lib = L
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(_ip)


def n_external(process: str) -> int:
    return lib().orc_n_external(process.encode())


def me2(process: str, par, p) -> float:
    """|M|^2 (averaged) of one event; p[n_ext,4] = (E,px,py,pz)."""
    par, pp = _d(par)
    p, ppp = _d(p)
    out = C.c_double()
    rc = lib().orc_me2(process.encode(), pp, ppp, C.byref(out))
    if rc != 0:
        raise ValueError(process)
    return out.value


def reweight(process: str, par_old, par_new, momenta, weights, nthreads: int = 0):
    """Eq. 3 on an SoA event set momenta[n_ext,4,n]. Returns (me_old, me_new, w_new, threads_used)."""
    momenta, pm = _d(momenta)
    weights, pw = _d(weights)
    n = weights.shape[0]
    assert momenta.shape == (n_external(process), 4, n)
    po, ppo = _d(par_old)
    pn, ppn = _d(par_new)
    a, b, w = np.empty(n), np.empty(n), np.empty(n)
    used = lib().orc_reweight(process.encode(), ppo, ppn, pm, pw, a.ctypes.data_as(_dp),
                              b.ctypes.data_as(_dp), w.ctypes.data_as(_dp), n, nthreads)
    if used < 0:
        raise ValueError(process)
    return a, b, w, used


def gamma(mu: int) -> np.ndarray:
    out = np.empty(32)
    lib().orc_gamma(mu, out.ctypes.data_as(_dp))
    return out.view(np.complex128).reshape(4, 4)


def spinor(kind: str, p, m: float, lam: int) -> np.ndarray:
    p, pp = _d(p)
    out = np.empty(8)
    lib().orc_spinor(0 if kind == "u" else 1, pp, float(m), int(lam), out.ctypes.data_as(_dp))
    return out.view(np.complex128)


def polvec(p, lam: int) -> np.ndarray:
    p, pp = _d(p)
    out = np.empty(8)
    lib().orc_polvec(pp, int(lam), out.ctypes.data_as(_dp))
    return out.view(np.complex128)


def colour_matrix(n: int) -> np.ndarray:
    f = math.factorial(n)
    out = np.empty((f, f))
    assert lib().orc_colour_matrix(n, out.ctypes.data_as(_dp)) == 0
    return out


def fabc() -> np.ndarray:
    out = np.empty((8, 8, 8))
    lib().orc_fabc(out.ctypes.data_as(_dp))
    return out


def jamps(n: int, par, p, hel, eps_override=None) -> np.ndarray:
    par, pp = _d(par)
    p, ppp = _d(p)
    hel, ph = _i(hel)
    out = np.empty(2 * math.factorial(n))
    if eps_override is not None:
        eo = np.ascontiguousarray(eps_override, dtype=np.complex128).reshape(n, 4)
        peo = eo.view(np.float64).ctypes.data_as(_dp)
    else:
        peo = None
    lib().orc_jamps(n, pp, ppp, ph, peo, out.ctypes.data_as(_dp))
    return out.view(np.complex128)


def me2_hel(n: int, par, p, hel, route: str = "F") -> float:
    par, pp = _d(par)
    p, ppp = _d(p)
    hel, ph = _i(hel)
    out = C.c_double()
    lib().orc_me2_hel(n, pp, ppp, ph, 0 if route == "F" else 1, C.byref(out))
    return out.value


def amp_epem(par, p, hel) -> complex:
    par, pp = _d(par)
    p, ppp = _d(p)
    hel, ph = _i(hel)
    out = np.empty(2)
    lib().orc_amp_epem(pp, ppp, ph, out.ctypes.data_as(_dp))
    return complex(out[0], out[1])


def cross_section(weights) -> float:
    """eq. 2: sigma ~ sum_k W_k, the plain left-to-right sum."""
    w, pw = _d(weights)
    return lib().orc_cross_section(pw, w.shape[0])


def me2_hel_qq(ng: int, par, p, hel, eps_override=None) -> float:
    """Colour-summed |M_h|^2 (no averaging) of q qbar -> t tbar (ng = 0) or q qbar -> t tbar g (ng = 1); p[4+ng,4], hel[4+ng] = +-1."""
    par, pp = _d(par)
    p, ppp = _d(p)
    hel, ph = _i(hel)
    out = C.c_double()
    if eps_override is not None:
        eo = np.ascontiguousarray(eps_override, dtype=np.complex128).reshape(4)
        peo = eo.view(np.float64).ctypes.data_as(_dp)
    else:
        peo = None
    assert lib().orc_me2_hel_qq(ng, pp, ppp, ph, peo, C.byref(out)) == 0
    return out.value


def denominator(n: int) -> float:
    return lib().orc_denominator(n)


def amp_epem_ng(n: int, par, p, hel, eps_override=None) -> complex:
    """Helicity amplitude iM of e+ e- -> n photons (PAPER.md:72-77 for n = 5); p[n+2,4], hel[n+2] = +-1."""
    par, pp = _d(par)
    p, ppp = _d(p)
    hel, ph = _i(hel)
    out = np.empty(2)
    if eps_override is not None:
        eo = np.ascontiguousarray(eps_override, dtype=np.complex128).reshape(n, 4)
        peo = eo.view(np.float64).ctypes.data_as(_dp)
    else:
        peo = None
    lib().orc_amp_epem_ng(n, pp, ppp, ph, peo, out.ctypes.data_as(_dp))
    return complex(out[0], out[1])
