"""Pins of the oracle's e+ e- -> n photons (Table 1: the paper's measured process is n = 5) against
things other than itself: textbook closed forms at n = 2, 3, the soft-photon (eikonal) theorem that ties the
normalisation of n + 1 photons to n photons up to n = 5, gauge invariance of every helicity amplitude, Lorentz
invariance, helicity selection rules, and the exact coupling scaling the paper's reweighting relies on.  CPU only."""
import math

import numpy as np
import pytest

import oracle as orc
from paper_2312_07440_b200 import events as ev
from test_oracle_pins import boost, mdot, rotation

P0 = ev.params()
E2 = 4.0 * math.pi * P0[0]


def events(n_photons, n):
    c = ev.photon_config(n_photons)
    m, _ = ev.generate(c, n)
    return c, [np.ascontiguousarray(m[:, :, k]) for k in range(n)]


def test_two_photon_textbook_closed_form():
    # (1/4) sum |M|^2 = 2 e^4 (u/t + t/u) for massless e+ e- -> gamma gamma; with the 1/2! of identical photons: e^4 (u/t + t/u)
    c, evs = events(2, 8)
    for p in evs:
        t, u = -2.0 * mdot(p[1], p[2]), -2.0 * mdot(p[1], p[3])
        assert orc.me2(c.process, P0, p) == pytest.approx(E2 ** 2 * (u / t + t / u), rel=1e-12)


def test_three_photon_closed_form():
    # massless e+ e- -> 3 gamma (Berends, Kleiss et al.): (1/4) sum |M|^2 = e^6 s sum_i a_i b_i (a_i^2 + b_i^2) / prod_i a_i b_i,
    # a_i = p1.k_i, b_i = p2.k_i; me2 carries the extra 1/3!
    c, evs = events(3, 8)
    for p in evs:
        a = [mdot(p[0], p[2 + j]) for j in range(3)]
        b = [mdot(p[1], p[2 + j]) for j in range(3)]
        s = 2.0 * mdot(p[0], p[1])
        cf = E2 ** 3 * s * sum(a[j] * b[j] * (a[j] ** 2 + b[j] ** 2) for j in range(3)) / np.prod(a) / np.prod(b)
        assert orc.me2(c.process, P0, p) == pytest.approx(cf / 6.0, rel=1e-11)


@pytest.mark.parametrize("n", [2, 3, 4])
def test_soft_photon_theorem_links_n_plus_one_to_n(n):
    # k -> 0:  sum|M_{n+1}|^2 -> e^2 (2 p1.p2) / ((p1.k)(p2.k)) sum|M_n|^2, i.e. me2_{n+1} -> eik * me2_n / (n + 1):
    # carries the closed-form normalisation of n = 2, 3 up to n = 5 (vertex factor, propagator, 1/n!)
    c, evs = events(n, 2)
    rng = np.random.default_rng(5 + n)
    for p in evs:
        d = rng.normal(size=3)
        d[2] *= 0.3
        d /= np.linalg.norm(d)
        eps = 2e-6 * c.sqrts
        k = np.array([eps, *(eps * d)])
        # exact momentum conservation (the eikonal pole IS the propagator next to the soft emission): rescale and boost
        # the n hard photons so that they recoil against k
        mrec = math.sqrt((c.sqrts - eps) ** 2 - eps ** 2)
        hard = boost(p[2:] * (mrec / c.sqrts), -k[1:] / (c.sqrts - eps))
        q = np.vstack([p[:2], hard, k])
        assert np.abs(q[2:].sum(axis=0) - q[:2].sum(axis=0)).max() < 1e-11 * c.sqrts
        eik = E2 * 2.0 * mdot(q[0], q[1]) / (mdot(q[0], k) * mdot(q[1], k))
        lhs = orc.me2("epem_" + "a" * (n + 1), P0, q)
        rhs = eik * orc.me2(c.process, P0, p) / (n + 1)
        assert lhs == pytest.approx(rhs, rel=2e-4)


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_gauge_invariance_of_every_helicity_amplitude(n):
    c, evs = events(n, 1)
    p = evs[0]
    rng = np.random.default_rng(n)
    scale = abs(orc.amp_epem_ng(n, P0, p, [-1, 1] + [1, -1, 1, -1, -1][:n]))
    assert scale > 0
    for trial in range(3 if n == 5 else 6):
        hel = [-1, 1] + list(rng.choice([-1, 1], size=n))
        j = int(rng.integers(n))
        eps = np.array([np.conj(orc.polvec(p[2 + i], hel[2 + i])) for i in range(n)])
        eps[j] = p[2 + j]                      # eps_j -> k_j
        assert abs(orc.amp_epem_ng(n, P0, p, hel, eps)) < 1e-10 * scale * c.sqrts
        # the override path reproduces the ordinary amplitude when given the ordinary polarisation vectors
        eps[j] = np.conj(orc.polvec(p[2 + j], hel[2 + j]))
        assert orc.amp_epem_ng(n, P0, p, hel, eps) == pytest.approx(orc.amp_epem_ng(n, P0, p, hel), rel=1e-13, abs=1e-30)


@pytest.mark.parametrize("n", [2, 3, 4])
def test_helicity_selection_parity_and_all_plus(n):
    c, evs = events(n, 1)
    p = evs[0]
    ref = abs(orc.amp_epem_ng(n, P0, p, [-1, 1] + [1, -1, 1, -1][:n]))
    assert ref > 0
    for lam in (-1, 1):                        # massless line: equal e+ and e- helicities give zero
        assert abs(orc.amp_epem_ng(n, P0, p, [lam, lam] + [1, -1, 1, -1][:n])) < 1e-13 * max(ref, 1e-300) + 1e-30
    # all photons with the same helicity: the tree amplitude vanishes
    for lam in (-1, 1):
        assert abs(orc.amp_epem_ng(n, P0, p, [-1, 1] + [lam] * n)) < 1e-10 * ref
    rng = np.random.default_rng(11 * n)
    for _ in range(4):                         # parity: flipping every helicity keeps |M_h|
        hel = [-1, 1] + list(rng.choice([-1, 1], size=n))
        a, b = abs(orc.amp_epem_ng(n, P0, p, hel)), abs(orc.amp_epem_ng(n, P0, p, [-h for h in hel]))
        assert a == pytest.approx(b, rel=1e-10, abs=1e-12 * ref)


@pytest.mark.parametrize("n", [2, 3, 4])
def test_boost_and_rotation_invariance(n):
    c, evs = events(n, 2)
    rng = np.random.default_rng(n)
    for p in evs:
        ref = orc.me2(c.process, P0, p)
        assert orc.me2(c.process, P0, boost(p, np.array([0.2, -0.3, 0.4]))) == pytest.approx(ref, rel=1e-10)
        R = rotation(rng)
        q = p.copy()
        q[:, 1:] = p[:, 1:] @ R.T
        assert orc.me2(c.process, P0, q) == pytest.approx(ref, rel=1e-11)


def test_five_photon_coupling_scaling_is_exact():
    # PAPER.md:77 (Table 1 caption): the reweighting of the paper changes the electroweak coupling only, so the
    # weight ratio of eq. 3 is (alpha'/alpha)^5 for every event
    c, evs = events(5, 2)
    for p in evs:
        a, b = orc.me2(c.process, c.params_old, p), orc.me2(c.process, c.params_new, p)
        assert a > 0 and b / a == pytest.approx((c.params_new[0] / c.params_old[0]) ** 5, rel=1e-13)
    m, w = ev.generate(c, 3)
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, m, w)
    assert np.array_equal(wn, w * (b / a))


def test_five_photon_rotation_invariance():
    c, evs = events(5, 1)
    p = evs[0]
    R = rotation(np.random.default_rng(3))
    q = p.copy()
    q[:, 1:] = p[:, 1:] @ R.T
    assert orc.me2(c.process, P0, q) == pytest.approx(orc.me2(c.process, P0, p), rel=1e-10)
