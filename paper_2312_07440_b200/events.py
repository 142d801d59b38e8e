"""Seeded synthetic event sets for the five BASELINE.json configs (+ the paper's own e+e- -> 5 gamma, + q qbar -> t tbar (g)).

This module is the ONLY code shared by the CPU oracle (tests / cpu_baseline) and
the CUDA path.  It holds none of the method's arithmetic (no wavefunctions,
vertices, colour, |M|^2): it only draws phase-space points and weights, as
SURVEY.md §8(d) D1 prescribes, standing in for the LHE event files the paper
parses (PAPER.md:87 step 2), which do not exist here.

Recipe (all host-side numpy, FP64):
  * PRNG: counter-based splitmix64; uniform k of a stream is
    u_k = ((mix(seed + (k+1)*GOLDEN) >> 11) + 0.5) / 2^53  in (0,1).
  * candidate event c of a config consumes the R = 4*n_final + 2 uniforms with
    counters [c*R, (c+1)*R): 4 per final-state particle for RAMBO, 2 for the
    Box-Muller normal that gives the weight W = exp(z).
  * beams: leg 0 = (rs/2,0,0,+rs/2), leg 1 = (rs/2,0,0,-rs/2).
  * final state: RAMBO flat phase space (Kleiss, Stirling, Ellis), massive
    legs by the usual xi-rescaling solved with Newton; a final polish makes
    sum(p_vec)=0 exactly and sum(E)=sqrts to rounding with every leg on shell.
  * cuts: every extra gluon pT > 20 GeV; cfgs 4,5 also Delta R > 0.4 between
    every pair of extra gluons.  Rejected candidates are skipped; the first
    n accepted candidates (in counter order) are the events.
Layout returned: momenta[n_ext, 4, n_events] (E,px,py,pz) C-contiguous float64
(= the SoA `momenta[(ip*4+mu)*n + ievt]` of include/rwgt.h), weights[n_events].
"""
from __future__ import annotations

import dataclasses
import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

# parameter vector order == struct rwgt_params in include/rwgt.h
PARAM_NAMES = ("alpha_em", "alpha_s", "mZ", "GammaZ", "sin2_thetaW", "mt",
               "Gamma_t", "ggg_scale", "gggg_scale")


def params(**kw) -> np.ndarray:
    base = dict(alpha_em=1.0 / 132.5, alpha_s=0.118, mZ=91.1876, GammaZ=2.4952,
                sin2_thetaW=0.2312, mt=173.0, Gamma_t=0.0, ggg_scale=1.0,
                gggg_scale=1.0)
    base.update(kw)
    return np.array([base[k] for k in PARAM_NAMES], dtype=np.float64)


@dataclasses.dataclass(frozen=True)
class Config:
    index: int            # 1..5 as in SURVEY.md §8
    process: str          # name understood by rwgt_create and by the oracle
    n_events: int
    sqrts: float
    final_masses: tuple   # masses of the final-state legs, in leg order
    n_extra_gluons: int   # number of trailing final-state legs the pT / Delta R cuts apply to
    dr_cut: bool
    seed: int
    params_old: np.ndarray
    params_new: np.ndarray
    precisions: tuple

    @property
    def n_ext(self) -> int:
        return 2 + len(self.final_masses)


_KAPPA = 0.1
_MT = 173.0
CONFIGS = (
    Config(1, "epem_mupmum", 16384, 500.0, (0.0, 0.0), 0, False, 20231207 + 1,
           params(), params(GammaZ=2.60, sin2_thetaW=0.235), ("fp64",)),
    Config(2, "gg_ttx", 1048576, 1500.0, (_MT, _MT), 0, False, 20231207 + 2,
           params(), params(ggg_scale=1 + _KAPPA), ("fp64",)),
    Config(3, "gg_ttxg", 1048576, 1500.0, (_MT, _MT, 0.0), 1, False, 20231207 + 3,
           params(), params(ggg_scale=1 + _KAPPA, gggg_scale=1 + _KAPPA),
           ("fp64", "fp32")),
    Config(4, "gg_ttxgg", 262144, 1500.0, (_MT, _MT, 0.0, 0.0), 2, True, 20231207 + 4,
           params(), params(ggg_scale=1 + _KAPPA, gggg_scale=1 + _KAPPA),
           ("fp64", "fp32")),
    Config(5, "gg_ttxggg", 65536, 1500.0, (_MT, _MT, 0.0, 0.0, 0.0), 3, True, 20231207 + 5,
           params(), params(ggg_scale=1 + _KAPPA, gggg_scale=1 + _KAPPA),
           ("fp64", "fp32")),
    # Not a BASELINE.json config: the process the paper itself measured (Table 1:
    # e+ e- -> 5 gamma, SM, the electroweak coupling re-drawn per reweight iteration).
    # 2^17 events stand in for the "10^5 events" of the paper's Fig. 3; sqrt(s) and the
    # cuts are not stated in the paper: 500 GeV as cfg 1, every photon pT > 20 GeV and Delta R > 0.4.
    Config(6, "epem_aaaaa", 131072, 500.0, (0.0,) * 5, 5, True, 20231207 + 6,
           params(), params(alpha_em=1.0 / 128.0), ("fp64",)),
    # Not BASELINE.json configs: structurally different amplitudes for the final states of cfgs 2 and 3 (PAPER.md:87 last
    # sentence, "LO multiprocesses"): a massless quark-antiquark pair instead of the two gluons.  Same sqrt(s), masses and
    # cuts as cfgs 2 / 3; q qbar -> t tbar has no gluon self-coupling, so its new set changes alpha_s (a running-coupling style change).
    Config(7, "qqx_ttx", 1048576, 1500.0, (_MT, _MT), 0, False, 20231207 + 7,
           params(), params(alpha_s=0.108), ("fp64",)),
    Config(8, "qqx_ttxg", 1048576, 1500.0, (_MT, _MT, 0.0), 1, False, 20231207 + 8,
           params(), params(ggg_scale=1 + _KAPPA, gggg_scale=1 + _KAPPA), ("fp64",)),
)


def photon_config(n_photons: int, n_events: int = 4096) -> Config:
    """e+ e- -> n photons, n = 2..5 (n = 5 is config 6; the others are parity-test cases)."""
    if n_photons == 5:
        return dataclasses.replace(CONFIGS[5], n_events=n_events)
    return Config(60 + n_photons, "epem_" + "a" * n_photons, n_events, 500.0, (0.0,) * n_photons,
                  n_photons, True, 20231207 + 60 + n_photons, params(), params(alpha_em=1.0 / 128.0), ("fp64",))


def config(index_or_process) -> Config:
    for c in CONFIGS:
        if c.index == index_or_process or c.process == index_or_process:
            return c
    raise KeyError(index_or_process)


# ---------------------------------------------------------------------------- named lists of new parameter sets (inputs only)
# PAPER.md:87 step 7 / Fig. 3: K new sets per pass.  The lists below are what bench.py times with K > 1 and what
# tests/golden/make_goldens.py --sets evaluates with the oracle; they are inputs (numbers typed in), no arithmetic of the method.
KSET_LISTS = ("bench4", "bench8", "bench16", "general4", "mass4")
# which lists each config stores oracle values for (tests/golden/ksets_cfg<N>_<list>.npz)
KSET_GOLDENS = {3: ("bench8", "mass4"), 4: ("bench8", "general4", "mass4"), 5: ("bench4", "bench16", "general4", "mass4")}


def kset_list(cfg: "Config", name: str) -> list:
    """bench<K>: the coupling-only 'diagonal' lists bench.py times (ggg_scale = gggg_scale = 1 + 0.1 (k+1) / K: polynomial mode at
    n >= 4, one level pass at n = 3); general4: independent three- and four-gluon scales with the old set among them (rank above
    the diagonal case); mass4: other top masses (externals and denominators redone per set), the config's new set and the old set."""
    if name.startswith("bench"):
        K = int(name[5:])
        return [params(ggg_scale=1 + 0.1 * (k + 1) / K, gggg_scale=1 + 0.1 * (k + 1) / K) for k in range(K)]
    if name == "general4":
        return [params(ggg_scale=1.1, gggg_scale=0.9), params(ggg_scale=0.95, gggg_scale=1.2), cfg.params_old.copy(),
                params(ggg_scale=1.2, gggg_scale=1.05, alpha_s=0.125)]
    if name == "mass4":
        return [params(mt=170.0, ggg_scale=1.1, gggg_scale=1.1), cfg.params_new.copy(), params(mt=176.5, ggg_scale=0.9), cfg.params_old.copy()]
    raise KeyError(name)


def kset_sample(cfg: "Config") -> np.ndarray:
    """Event indices of the config's full seeded set on which the K-set goldens are stored: a contiguous prefix longer than two
    rounds of a persistent one-CTA-per-SM launch (148 CTAs x at most 32 / 8 / 2 events in flight per CTA for 3 / 4 / 5 gluons), every
    stride-th event of the rest (every later round of the launch is hit) and the last events (the ragged tail)."""
    n = cfg.n_events
    prefix, strided, tail = {3: (12288, 2048, 256), 4: (2560, 512, 64), 5: (304, 96, 16)}[cfg.index]
    rest = np.linspace(prefix, n - tail - 1, strided).astype(np.int64)
    return np.unique(np.concatenate([np.arange(prefix), rest, np.arange(n - tail, n)]))


def _splitmix64(counter: np.ndarray, seed: int) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = np.uint64(seed) + (counter.astype(np.uint64) + np.uint64(1)) * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniforms(seed: int, start: int, count: int) -> np.ndarray:
    k = np.arange(start, start + count, dtype=np.uint64)
    z = _splitmix64(k, seed)
    return ((z >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def _rambo(u: np.ndarray, sqrts: float, masses) -> np.ndarray:
    """u[c, i, 4] uniforms -> p[c, i, 4] (E,px,py,pz) summing to (sqrts,0,0,0)."""
    nf = len(masses)
    c = 2.0 * u[:, :, 0] - 1.0
    phi = 2.0 * np.pi * u[:, :, 1]
    q0 = -np.log(u[:, :, 2] * u[:, :, 3])
    st = np.sqrt(np.maximum(0.0, 1.0 - c * c))
    q = np.stack([q0, q0 * st * np.cos(phi), q0 * st * np.sin(phi), q0 * c], axis=2)
    Q = q.sum(axis=1)
    M = np.sqrt(Q[:, 0] ** 2 - Q[:, 1] ** 2 - Q[:, 2] ** 2 - Q[:, 3] ** 2)
    b = -Q[:, 1:] / M[:, None]
    x = sqrts / M
    g = Q[:, 0] / M
    a = 1.0 / (1.0 + g)
    bq = np.einsum("ck,cik->ci", b, q[:, :, 1:])
    p = np.empty_like(q)
    p[:, :, 0] = x[:, None] * (g[:, None] * q[:, :, 0] + bq)
    p[:, :, 1:] = x[:, None, None] * (q[:, :, 1:] + b[:, None, :] * q[:, :, 0:1]
                                      + (a[:, None] * bq)[:, :, None] * b[:, None, :])
    # Polish (not part of RAMBO proper, it only removes rounding noise that the
    # boost amplifies for a few candidates): make the 3-momenta sum to zero
    # exactly, then fix the common scale xi so the on-shell energies sum to sqrts.
    m = np.asarray(masses, dtype=np.float64)
    m2 = (m * m)[None, :]
    p[:, -1, 1:] = -p[:, :-1, 1:].sum(axis=1)
    p2 = np.sum(p[:, :, 1:] ** 2, axis=2)
    xi = np.full(p.shape[0], np.sqrt(1.0 - (m.sum() / sqrts) ** 2))
    for _ in range(60):
        e = np.sqrt(m2 + (xi * xi)[:, None] * p2)
        f = e.sum(axis=1) - sqrts
        df = (xi[:, None] * p2 / e).sum(axis=1)
        step = f / df
        xi = xi - step
        if np.max(np.abs(step) / xi) < 1e-15:
            break
    p[:, :, 1:] *= xi[:, None, None]
    p[:, :, 0] = np.sqrt(m2 + np.sum(p[:, :, 1:] ** 2, axis=2))
    return p


def _passes_cuts(p: np.ndarray, n_extra: int, dr_cut: bool) -> np.ndarray:
    ok = np.ones(p.shape[0], dtype=bool)
    if n_extra == 0:
        return ok
    g = p[:, -n_extra:, :]
    pt = np.hypot(g[:, :, 1], g[:, :, 2])
    ok &= np.all(pt > 20.0, axis=1)
    if dr_cut and n_extra > 1:
        y = 0.5 * np.log((g[:, :, 0] + g[:, :, 3]) / (g[:, :, 0] - g[:, :, 3]))
        ph = np.arctan2(g[:, :, 2], g[:, :, 1])
        for i in range(n_extra):
            for j in range(i + 1, n_extra):
                dphi = np.abs(ph[:, i] - ph[:, j])
                dphi = np.where(dphi > np.pi, 2.0 * np.pi - dphi, dphi)
                dr = np.hypot(y[:, i] - y[:, j], dphi)
                ok &= dr > 0.4
    return ok


def generate(cfg: Config, n_events: int | None = None, seed: int | None = None,
             first_candidate: int = 0):
    """Return (momenta[n_ext,4,n], weights[n]) for the first n accepted candidates."""
    n = cfg.n_events if n_events is None else int(n_events)
    seed = cfg.seed if seed is None else int(seed)
    nf = len(cfg.final_masses)
    R = 4 * nf + 2
    mom = np.empty((cfg.n_ext, 4, n), dtype=np.float64)
    wts = np.empty(n, dtype=np.float64)
    half = 0.5 * cfg.sqrts
    mom[0] = np.array([half, 0.0, 0.0, half])[:, None]
    mom[1] = np.array([half, 0.0, 0.0, -half])[:, None]
    filled, cand = 0, first_candidate
    while filled < n:
        block = max(1024, int((n - filled) * 1.15) + 64)
        u = uniforms(seed, cand * R, block * R).reshape(block, R)
        cand += block
        p = _rambo(u[:, : 4 * nf].reshape(block, nf, 4), cfg.sqrts, cfg.final_masses)
        ok = _passes_cuts(p, cfg.n_extra_gluons, cfg.dr_cut)
        z = np.sqrt(-2.0 * np.log(u[:, 4 * nf])) * np.cos(2.0 * np.pi * u[:, 4 * nf + 1])
        p, z = p[ok], z[ok]
        take = min(n - filled, p.shape[0])
        mom[2:, :, filled:filled + take] = np.transpose(p[:take], (1, 2, 0))
        wts[filled:filled + take] = np.exp(z[:take])
        filled += take
    return np.ascontiguousarray(mom), wts
