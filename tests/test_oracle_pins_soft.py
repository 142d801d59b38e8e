"""Soft-gluon pins of the oracle for g g -> t tbar + gluons with n = 3, 4, 5 gluons in total (SURVEY.md C9,
lines 454-455: the (n-2)! of the averaging denominator and the absolute scale at n = 4, 5 had no pin other than the oracle's own
rule restated).  PAPER.md:66 names the helicity-amplitude method and prints no formula, so the pin is the soft-gluon theorem, which
ties the (n)-gluon amplitudes to the (n-1)-gluon ones and so, step by step, to the closed form of g g -> t tbar (n = 2, Ellis /
Stirling / Webber table 10.2, test_oracle_pins.py) and the worked point of g g -> t tbar g (tests/golden/c10c_gg_ttxg.txt).

Colour-ordered form (Berends, Giele Nucl. Phys. B306 (1988) 759; Mangano, Parke Phys. Rept. 200 (1991) 301, sect. 3.4): when gluon s
with momentum k and polarisation eps becomes soft, the amplitude of the ordering  t, sigma_1 ... sigma_n, tbar  factorises as
        J_sigma(n)  ->  -g_s ( eps.p_a / p_a.k  -  eps.p_b / p_b.k )  J_{sigma without s}(n-1),
a and b being the neighbours of s in the ordering (the top at the left end, the antitop at the right end, massive or not).  The
overall -1 is the phase convention of the oracle's vertices; |M|^2 does not see it.  Squared, summed over the soft gluon's
polarisations (sum eps^mu eps^nu* -> -g^{mu nu}; the gauge terms drop out of the colour-summed square) and over colours with the
n-gluon colour matrix C_n, and averaged:
        |M_n|^2  ->  g_s^2  [ sum_h J'^dagger (C_n o E) J' ] / [ sum_h J'^dagger C_{n-1} J' ]  x  |M_{n-1}|^2 / (k+1),
        E[sigma, sigma'] = - (v_a - v_b).(v_a' - v_b'),   v_i = p_i / (p_i.k),
where J' are the (n-1)-gluon amplitudes, sigma -> sigma without s maps the rows of C_n onto those of C_{n-1}, and k+1 is the number of
identical final-state gluons of the n-gluon process: its identical-particle factor is 1/(k+1)!, that of the (n-1)-gluon process
1/k!.  An averaging denominator at n = 4 or 5 that is not 256 (n-2)!, a wrong overall factor in the four- or five-gluon currents, or a
colour matrix C_n that does not reduce to C_{n-1}, fails here.  Everything in this file is CPU-only and uses the oracle alone."""
import itertools
import math

import numpy as np
import pytest

import oracle as orc
from paper_2312_07440_b200 import events as ev


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def leg_of_gluon(j):
    """legs are [g, g, t, tbar, g...]: gluon label j sits on leg j (incoming) or j + 2 (outgoing)"""
    return j if j < 2 else j + 2


def born_event(n_born, k=3):
    """event k of the seeded set of the config with n_born gluons (cfg index == number of gluons for the g g processes)"""
    c = ev.config(n_born)
    m, _ = ev.generate(c, k + 1)
    return c, np.ascontiguousarray(m[:, :, k])


def soft_momentum(rng, w):
    d = rng.normal(size=3)
    d /= np.linalg.norm(d)
    return w * np.array([1.0, *d])


def with_soft_gluon(pb, k):
    """(n+1)-leg event: the Born event pb with the soft gluon k appended and the Born final state taking the recoil, every leg on
    its mass shell and the momentum sum exact.  The oracle forms the top propagators from the antitop's side, so the last one is
    1 / ((p_t + k)^2 - m_t^2) only if momentum is conserved: appending k to an unchanged Born event would make it 1 / 0.
    The Born final state (at rest, invariant mass sqrt(s)) has its three-momenta scaled by a common factor until its invariant mass
    is that of Q - k, and is then boosted to the total momentum Q - k; it moves by O(k) and the beams stay as they are."""
    fin = pb[2:].copy()
    Q = pb[0] + pb[1]
    assert np.allclose(Q[1:], 0, atol=1e-9 * Q[0]) and np.allclose(fin.sum(axis=0), Q, atol=1e-9 * Q[0])
    m2 = np.maximum(0.0, fin[:, 0] ** 2 - (fin[:, 1:] ** 2).sum(axis=1))
    pabs2 = (fin[:, 1:] ** 2).sum(axis=1)
    P = Q - k
    M = math.sqrt(mdot(P, P))
    xi = 1.0
    for _ in range(50):                                              # Newton on sum_i sqrt(m_i^2 + xi^2 |p_i|^2) = M
        e = np.sqrt(m2 + xi * xi * pabs2)
        xi -= (e.sum() - M) / (xi * pabs2 / e).sum()
    e = np.sqrt(m2 + xi * xi * pabs2)
    rest = np.column_stack([e, xi * fin[:, 1:]])
    beta, gamma = P[1:] / P[0], P[0] / M
    bp = rest[:, 1:] @ beta
    b2 = beta @ beta
    out = np.empty_like(rest)
    out[:, 0] = gamma * (rest[:, 0] + bp)
    out[:, 1:] = rest[:, 1:] + np.outer((gamma - 1) * bp / b2 + gamma * rest[:, 0], beta)
    p = np.vstack([pb[:2], out, k])
    assert np.abs(p[:2].sum(axis=0) - p[2:].sum(axis=0)).max() < 1e-11 * Q[0]
    return p


def neighbours(sigma, s):
    """legs left and right of gluon s in the ordering t, sigma..., tbar"""
    pos = sigma.index(s)
    left = 2 if pos == 0 else leg_of_gluon(sigma[pos - 1])
    right = 3 if pos == len(sigma) - 1 else leg_of_gluon(sigma[pos + 1])
    return left, right


@pytest.mark.parametrize("n", [3, 4, 5])
def test_every_colour_flow_amplitude_factorises_when_the_last_gluon_is_soft(n):
    c, pb = born_event(n - 1)
    par = c.params_old
    g = math.sqrt(4 * math.pi * par[1])
    perms_n = list(itertools.permutations(range(n)))
    perms_b = list(itertools.permutations(range(n - 1)))
    s = n - 1
    rng = np.random.default_rng(100 + n)
    # size of a typical (n-1)-gluon amplitude: for helicities whose Born amplitudes vanish the leading soft term is zero and only
    # the non-singular remainder is left, so the bound is set by the largest amplitudes of the event, not by the configuration's own
    j_typ = max(np.abs(orc.jamps(n - 1, par, pb, h)).max() for h in itertools.product((1, -1), repeat=n + 1))
    for _ in range(3):
        hel_b = rng.choice([-1, 1], size=n + 1)
        Jb = orc.jamps(n - 1, par, pb, hel_b)
        for w in (1e-2, 1e-4):                                       # soft gluon energy in GeV; corrections are O(w / m_t)
            k = soft_momentum(rng, w)
            p = with_soft_gluon(pb, k)
            v = [p[l] / mdot(p[l], k) for l in range(n + 1)]
            for hs in (1, -1):
                eps = orc.polvec(k, hs).conj()                       # outgoing gluon
                Jn = orc.jamps(n, par, p, np.concatenate([hel_b, [hs]]))
                pred, eik = np.empty(len(perms_n), dtype=complex), np.empty(len(perms_n), dtype=complex)
                for i, sigma in enumerate(perms_n):
                    a, b = neighbours(sigma, s)
                    rest = tuple(x for x in sigma if x != s)
                    eik[i] = -g * (mdot(eps, v[a]) - mdot(eps, v[b]))
                    pred[i] = eik[i] * Jb[perms_b.index(rest)]
                scale = np.abs(eik).max() * j_typ
                assert np.abs(Jn - pred).max() < 0.05 * w * scale, (n, w, hs, np.abs(Jn - pred).max() / scale)


def soft_prediction(n, par, pb, k):
    """g_s^2 [sum_h J'^dagger (C_n o E) J'] / [sum_h J'^dagger C_{n-1} J'] for the (n-1)-gluon event pb and the soft momentum k"""
    perms_n = list(itertools.permutations(range(n)))
    perms_b = list(itertools.permutations(range(n - 1)))
    s = n - 1
    p = with_soft_gluon(pb, k)
    v = [p[l] / mdot(p[l], k) for l in range(n + 1)]
    d = np.array([v[a] - v[b] for a, b in (neighbours(sigma, s) for sigma in perms_n)])          # [n!, 4]
    E = -(np.outer(d[:, 0], d[:, 0]) - d[:, 1:] @ d[:, 1:].T)
    red = np.array([perms_b.index(tuple(x for x in sigma if x != s)) for sigma in perms_n])
    CE = orc.colour_matrix(n) * E
    Cb = orc.colour_matrix(n - 1)
    num = den = 0.0
    for hel in itertools.product((1, -1), repeat=n + 1):
        Jb = orc.jamps(n - 1, par, pb, hel)
        Jx = Jb[red]
        num += np.vdot(Jx, CE @ Jx).real
        den += np.vdot(Jb, Cb @ Jb).real
    return 4 * math.pi * par[1] * num / den, den


@pytest.mark.parametrize("n,final_gluons", [(3, 1), (4, 2), (5, 3)])
def test_me2_soft_limit_fixes_the_identical_gluon_factor_and_the_scale(n, final_gluons):
    name = {2: "gg_ttx", 3: "gg_ttxg", 4: "gg_ttxgg", 5: "gg_ttxggg"}
    c, pb = born_event(n - 1)
    par = c.params_old
    born = orc.me2(name[n - 1], par, pb)
    rng = np.random.default_rng(200 + n)
    for trial in range(2 if n == 5 else 3):
        for w in (1e-2, 1e-4):
            k = soft_momentum(rng, w)
            ratio, den = soft_prediction(n, par, pb, k)
            # the colour sum of the (n-1)-gluon amplitudes over its averaging denominator is the oracle's own |M_{n-1}|^2:
            # the jamps / colour_matrix pair used above is the one me2 uses
            assert abs(den / orc.denominator(n - 1) / born - 1) < 1e-10
            got = orc.me2(name[n], par, with_soft_gluon(pb, k))
            want = ratio * born / final_gluons
            assert abs(got / want - 1) < 0.05 * w, (n, w, got / want)


def test_soft_limit_tells_a_wrong_identical_gluon_factor():
    """the pin has teeth: with k! replaced by 1 or by (k+1)! the n = 4 prediction is off by a factor 2, far outside the bound"""
    c, pb = born_event(3)
    par = c.params_old
    k = soft_momentum(np.random.default_rng(7), 1e-3)
    ratio, _ = soft_prediction(4, par, pb, k)
    got = orc.me2("gg_ttxgg", par, with_soft_gluon(pb, k))
    born = orc.me2("gg_ttxg", par, pb)
    assert abs(got / (ratio * born / 2) - 1) < 1e-4
    assert abs(got / (ratio * born / 1) - 1) > 0.4 and abs(got / (ratio * born / 6) - 1) > 0.4
