"""Pins of the oracle's q qbar -> t tbar and q qbar -> t tbar g (a structurally different amplitude for the final
states of cfgs 2 / 3) against things other than itself: the textbook closed form of q qbar -> Q Qbar, gauge invariance, Lorentz
invariance, parity, helicity selection on the massless line, and the soft-gluon limit, whose colour correlations are evaluated
here from Gell-Mann matrices typed into this file.  CPU only."""
import itertools
import math

import numpy as np
import pytest

import oracle as orc
from paper_2312_07440_b200 import events as ev
from test_oracle_pins import boost, rotation, mdot


def event(idx, k):
    c = ev.config(idx)
    m, _ = ev.generate(c, k + 1)
    return c, np.ascontiguousarray(m[:, :, k])


def test_qqx_ttx_textbook_closed_form():
    """Ellis, Stirling, Webber, QCD and Collider Physics, table 10.2: averaged |M|^2 (q qbar -> Q Qbar) = g^4 (4/9)(tau1^2 + tau2^2 + rho/2),
    tau_i = 2 p_i.p_Q / s, rho = 4 m^2 / s.  Also in a boosted and rotated frame, and for another mass / coupling."""
    rng = np.random.default_rng(1)
    for k in range(6):
        c, p = event(7, k)
        for par in (c.params_old, c.params_new, ev.params(alpha_s=0.2)):
            g4 = (4 * math.pi * par[1]) ** 2
            for q in (p, boost(p, np.array([0.3, -0.2, 0.4])), np.concatenate([p[:, :1], p[:, 1:] @ rotation(rng).T], axis=1)):
                s = mdot(q[0] + q[1], q[0] + q[1])
                t1, t2, rho = 2 * mdot(q[0], q[2]) / s, 2 * mdot(q[1], q[2]) / s, 4 * par[5] ** 2 / s
                assert abs(orc.me2("qqx_ttx", par, q) / (g4 * 4 / 9 * (t1 * t1 + t2 * t2 + rho / 2)) - 1) < 1e-12


def test_qqx_helicity_selection_and_parity():
    """Massless light line: equal q and qbar helicity labels give exactly zero; flipping every helicity keeps |M_h|^2 (both sets)."""
    for ng, idx in ((0, 7), (1, 8)):
        c, p = event(idx, 2)
        for par in (c.params_old, c.params_new):
            tot = 0.0
            for hel in itertools.product((1, -1), repeat=4 + ng):
                a = orc.me2_hel_qq(ng, par, p, hel)
                tot += a
                if hel[0] == hel[1]:
                    assert a == 0.0 or a < 1e-28 * max(1.0, tot)
                if hel[0] > 0:
                    b = orc.me2_hel_qq(ng, par, p, [-h for h in hel])
                    assert abs(a - b) <= 1e-11 * max(a, b) + 1e-30
            assert abs(tot / 36.0 / orc.me2(c.process, par, p) - 1) < 1e-13


def test_qqx_ttxg_gauge_invariance():
    """eps -> k sends every helicity's colour-summed |M_h|^2 to zero at kappa = 0; not once the ggg coupling is rescaled alone (Q1)."""
    c, p = event(8, 1)
    k = p[4] / np.abs(p[4]).max()
    for hel in itertools.product((1, -1), repeat=5):
        if hel[0] == hel[1]:
            continue
        ref = orc.me2_hel_qq(1, c.params_old, p, hel)
        assert orc.me2_hel_qq(1, c.params_old, p, hel, eps_override=k.astype(complex)) < 1e-22 * ref
    assert orc.me2_hel_qq(1, c.params_new, p, [1, -1, 1, 1, 1], eps_override=k.astype(complex)) > 1e-8 * ref


def test_qqx_ttxg_boost_old_rotation_both():
    rng = np.random.default_rng(3)
    c, p = event(8, 3)
    pb = boost(p, np.array([-0.25, 0.1, 0.35]))
    pr = p.copy()
    pr[:, 1:] = p[:, 1:] @ rotation(rng).T
    ro, rn = orc.me2(c.process, c.params_old, p), orc.me2(c.process, c.params_new, p)
    assert abs(orc.me2(c.process, c.params_old, pb) / ro - 1) < 1e-11
    assert abs(orc.me2(c.process, c.params_old, pr) / ro - 1) < 1e-11
    assert abs(orc.me2(c.process, c.params_new, pr) / rn - 1) < 1e-11
    assert abs(rn / ro - 1) > 1e-4                           # the ggg coupling enters
    # |M'|^2 is an exact quadratic in the ggg scale (one three-gluon vertex at most)
    ks = [0.8, 1.0, 1.3]
    vals = [orc.me2(c.process, ev.params(ggg_scale=x), p) for x in ks]
    coef = np.polyfit(ks, vals, 2)
    assert abs(np.polyval(coef, 1.7) / orc.me2(c.process, ev.params(ggg_scale=1.7), p) - 1) < 1e-10


def gell_mann():
    l = np.zeros((8, 3, 3), dtype=complex)
    l[0][0, 1] = l[0][1, 0] = 1
    l[1][0, 1], l[1][1, 0] = -1j, 1j
    l[2][0, 0], l[2][1, 1] = 1, -1
    l[3][0, 2] = l[3][2, 0] = 1
    l[4][0, 2], l[4][2, 0] = -1j, 1j
    l[5][1, 2] = l[5][2, 1] = 1
    l[6][1, 2], l[6][2, 1] = -1j, 1j
    l[7] = np.diag([1, 1, -2]) / math.sqrt(3)
    return l / 2


def test_qqx_ttxg_soft_gluon_limit():
    """Soft-gluon theorem (Bassetto, Ciafaloni, Marchesini; Catani, Seymour hep-ph/9605323 eq. 4.2 with massive legs):
        |M(q qbar -> t tbar g)|^2 -> - g^2 sum_{i,j} <T_i.T_j> p_i.p_j / ((p_i.k)(p_j.k)) |M(q qbar -> t tbar)|^2      (k -> 0)
    summed over all ordered pairs including i = j (T_i^2 = C_F, p_i^2 = m_i^2).  The Born amplitude has the single colour structure
    T^c_{ji} T^c_{kl}, so <T_i.T_j> are numbers; they are computed here from the generators above (colour conservation: every leg
    taken as outgoing, an incoming quark acts with -T^T, an incoming antiquark / outgoing quark with T).  This links the normalisation,
    the vertex factors and the averaging of the five-leg amplitude to the closed form of the four-leg one."""
    T = gell_mann()
    born = np.einsum("cji,ckl->jikl", T, T)                              # indices: qbar j, q i, t k, tbar l
    def act(leg, c, x):
        # colour charge T^c of leg acting on the Born tensor; outgoing-particle convention
        if leg == 0:   # incoming quark i  == outgoing antiquark: -T^c_{i' i} transposed
            return -np.einsum("im,jmkl->jikl", T[c].T, x)
        if leg == 1:   # incoming antiquark j == outgoing quark
            return np.einsum("jm,mikl->jikl", T[c], x)
        if leg == 2:   # outgoing top k
            return np.einsum("km,jiml->jikl", T[c], x)
        return -np.einsum("lm,jikm->jikl", T[c].T, x)                    # outgoing antitop l
    norm = np.vdot(born, born).real
    TT = np.zeros((4, 4))
    for a in range(4):
        for b in range(4):
            TT[a, b] = sum(np.vdot(act(a, c, born), act(b, c, born)) for c in range(8)).real / norm
    assert np.allclose(np.diag(TT), 4 / 3) and np.allclose(TT.sum(axis=1), 0, atol=1e-12)       # C_F and colour conservation
    c, p4 = event(7, 4)
    par = c.params_old
    g2 = 4 * math.pi * par[1]
    born_me = orc.me2("qqx_ttx", par, p4)
    rng = np.random.default_rng(9)
    for _ in range(3):
        n = rng.normal(size=3)
        n /= np.linalg.norm(n)
        for w in (1e-2, 1e-4):                                           # gluon energy in GeV; the correction is O(w / m_t)
            k = w * np.array([1.0, *n])
            p5 = np.vstack([p4, k])
            eik = 0.0
            for a in range(4):
                for b in range(4):
                    eik -= TT[a, b] * mdot(p4[a], p4[b]) / (mdot(p4[a], k) * mdot(p4[b], k))
            got = orc.me2("qqx_ttxg", par, p5)
            assert abs(got / (g2 * eik * born_me) - 1) < 0.01 * w, (w, got / (g2 * eik * born_me))
