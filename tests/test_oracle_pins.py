"""Pins of the CPU oracle against things other than itself (closed forms, identities,
invariances, brute force, SURVEY.md §8(c) worked values).  CPU only."""
import itertools
import math
import os

import numpy as np
import pytest

import oracle as orc
from paper_2312_07440_b200 import events as ev

GOLD = os.path.join(os.path.dirname(__file__), "golden")
G = np.diag([1.0, -1.0, -1.0, -1.0])


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def slash(a):
    return sum(G[mu, mu] * a[mu] * orc.gamma(mu) for mu in range(4))


def rand_mom(rng, m):
    p3 = rng.normal(size=3) * 200.0
    return np.array([math.sqrt(m * m + p3 @ p3), *p3])


def special_momenta(m):
    out = [np.array([math.sqrt(m * m + 9.0), 0.0, 0.0, 3.0]), np.array([math.sqrt(m * m + 9.0), 0.0, 0.0, -3.0]),
           np.array([math.sqrt(m * m + 25.0), 3.0, -4.0, 0.0])]
    if m > 0:
        out.append(np.array([m, 0.0, 0.0, 0.0]))
    return out


def boost(p, beta):
    """Boost the rows of p[...,4] by velocity vector beta."""
    b2 = beta @ beta
    g = 1.0 / math.sqrt(1.0 - b2)
    bp = p[..., 1:] @ beta
    out = np.empty_like(p)
    out[..., 0] = g * (p[..., 0] + bp)
    out[..., 1:] = p[..., 1:] + np.outer((g - 1.0) * bp / b2 + g * p[..., 0], beta).reshape(p[..., 1:].shape)
    return out


def rotation(rng):
    q, r = np.linalg.qr(rng.normal(size=(3, 3)))
    q = q @ np.diag(np.sign(np.diag(r)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def event_aos(cfg_index, k, n=None):
    c = ev.config(cfg_index)
    m, w = ev.generate(c, n or (k + 1))
    return c, np.ascontiguousarray(m[:, :, k])


# ------------------------------------------------------------------ gamma matrices, SU(3)
def test_clifford_algebra():
    for mu in range(4):
        for nu in range(4):
            ac = orc.gamma(mu) @ orc.gamma(nu) + orc.gamma(nu) @ orc.gamma(mu)
            assert np.allclose(ac, 2 * G[mu, nu] * np.eye(4), atol=1e-15)
        assert np.allclose(orc.gamma(5) @ orc.gamma(mu) + orc.gamma(mu) @ orc.gamma(5), 0, atol=1e-15)
    g5 = 1j * orc.gamma(0) @ orc.gamma(1) @ orc.gamma(2) @ orc.gamma(3)
    assert np.allclose(g5, orc.gamma(5), atol=1e-15)
    assert np.allclose(orc.gamma(0).conj().T, orc.gamma(0))


def test_structure_constants():
    f = orc.fabc()
    assert abs(f[0, 1, 2] - 1.0) < 1e-15
    assert abs(f[0, 3, 6] - 0.5) < 1e-15 and abs(f[2, 3, 4] - 0.5) < 1e-15
    assert abs(f[3, 4, 7] - math.sqrt(3) / 2) < 1e-15 and abs(f[5, 6, 7] - math.sqrt(3) / 2) < 1e-15
    assert np.allclose(f, -np.transpose(f, (1, 0, 2))) and np.allclose(f, np.transpose(f, (1, 2, 0)))
    # f^{acd} f^{bcd} = N delta^{ab}
    assert np.allclose(np.einsum("acd,bcd->ab", f, f), 3 * np.eye(8), atol=1e-14)


# ------------------------------------------------------------------ external wavefunctions (SURVEY C2 pins)
@pytest.mark.parametrize("m", [0.0, 173.0])
def test_spinors_dirac_equation_and_completeness(m):
    rng = np.random.default_rng(1)
    g0 = orc.gamma(0)
    for p in [rand_mom(rng, m) for _ in range(6)] + special_momenta(m):
        ps = slash(p)
        scale = p[0] ** 1.5
        su = np.zeros((4, 4), complex)
        sv = np.zeros((4, 4), complex)
        for lam in (+1, -1):
            u, v = orc.spinor("u", p, m, lam), orc.spinor("v", p, m, lam)
            assert np.abs((ps - m * np.eye(4)) @ u).max() < 1e-13 * scale
            assert np.abs((ps + m * np.eye(4)) @ v).max() < 1e-13 * scale
            su += np.outer(u, u.conj() @ g0)
            sv += np.outer(v, v.conj() @ g0)
            # normalisation ubar u = 2m, vbar v = -2m
            assert abs(u.conj() @ g0 @ u - 2 * m) < 1e-12 * p[0]
            assert abs(v.conj() @ g0 @ v + 2 * m) < 1e-12 * p[0]
            # helicity: (Sigma.p_hat) u = lam u, (Sigma.p_hat) v = -lam v, Sigma^i = gamma5 gamma0 gamma^i
            if p[1:] @ p[1:] > 0:
                ph = p[1:] / np.linalg.norm(p[1:])
                S = sum(ph[i] * orc.gamma(5) @ g0 @ orc.gamma(i + 1) for i in range(3))
                assert np.abs(S @ u - lam * u).max() < 1e-13 * math.sqrt(p[0] + m)
                assert np.abs(S @ v + lam * v).max() < 1e-13 * math.sqrt(p[0] + m)
        assert np.abs(su - (ps + m * np.eye(4))).max() < 1e-13 * p[0]
        assert np.abs(sv - (ps - m * np.eye(4))).max() < 1e-13 * p[0]


def test_polarisation_vectors():
    rng = np.random.default_rng(2)
    for p in [rand_mom(rng, 0.0) for _ in range(6)] + special_momenta(0.0):
        ph = p[1:] / np.linalg.norm(p[1:])
        comp = np.zeros((3, 3), complex)
        for lam in (+1, -1):
            e = orc.polvec(p, lam)
            assert e[0] == 0
            assert abs(mdot(e, p)) < 1e-13 * p[0]
            assert abs(mdot(e, e.conj()) + 1) < 1e-14
            assert abs(mdot(e, e)) < 1e-14
            assert np.abs(1j * np.cross(ph, e[1:]) - lam * e[1:]).max() < 1e-14
            comp += np.outer(e[1:], e[1:].conj())
        assert np.abs(comp - (np.eye(3) - np.outer(ph, ph))).max() < 1e-14
        # eps(-lam) = -eps(lam)^*
        assert np.abs(orc.polvec(p, -1) + orc.polvec(p, +1).conj()).max() < 1e-15


# ------------------------------------------------------------------ cfg 1
def epem_closed_form(par, p):
    a_em, _, mZ, GZ, sw2 = par[:5]
    e2 = 4 * math.pi * a_em
    cw2 = 1 - sw2
    gL, gR = -0.5 + sw2, sw2
    s = mdot(p[0] + p[1], p[0] + p[1])
    t = mdot(p[1] - p[3], p[1] - p[3])
    u = mdot(p[1] - p[2], p[1] - p[2])
    chi = s / (sw2 * cw2 * (s - mZ * mZ + 1j * mZ * GZ))
    A = lambda gi, gj: abs(1 + gi * gj * chi) ** 2
    return e2 * e2 / (s * s) * (u * u * (A(gL, gL) + A(gR, gR)) + t * t * (A(gL, gR) + A(gR, gL)))


def test_epem_closed_form_on_rambo_events():
    c = ev.config(1)
    m, _ = ev.generate(c, 40)
    for k in range(40):
        p = np.ascontiguousarray(m[:, :, k])
        for par in (c.params_old, c.params_new):
            assert abs(orc.me2(c.process, par, p) / epem_closed_form(par, p) - 1) < 2e-14


def test_epem_photon_only_limit_and_helicity_selection():
    c, p = event_aos(1, 3)
    # push the Z out of the picture: huge mass => pure QED 2 e^4 (t^2+u^2)/s^2
    par = ev.params(mZ=1e12)
    s = mdot(p[0] + p[1], p[0] + p[1])
    t = mdot(p[1] - p[3], p[1] - p[3])
    u = mdot(p[1] - p[2], p[1] - p[2])
    e4 = (4 * math.pi / 132.5) ** 2
    assert abs(orc.me2(c.process, par, p) / (2 * e4 * (t * t + u * u) / (s * s)) - 1) < 1e-12
    amps = {h: orc.amp_epem(c.params_old, p, h) for h in itertools.product((1, -1), repeat=4)}
    nz = [h for h, a in amps.items() if abs(a) > 1e-12]
    assert len(nz) == 4 and all(h[0] == -h[1] and h[2] == -h[3] for h in nz)


def test_epem_golden_worked_values():
    c = ev.config(1)
    for ct, old, new, ratio in np.loadtxt(os.path.join(GOLD, "c10a_epem_mupmum.txt")):
        st, h = math.sqrt(1 - ct * ct), 250.0
        # theta = angle(e-, mu-); e- is leg 1, along -z
        pm = np.array([h, h * st, 0.0, -h * ct])
        pp = np.array([h, -h * st, 0.0, h * ct])
        p = np.array([[h, 0, 0, h], [h, 0, 0, -h], pp, pm])
        a, b = orc.me2(c.process, c.params_old, p), orc.me2(c.process, c.params_new, p)
        assert abs(a / old - 1) < 1e-13 and abs(b / new - 1) < 1e-13 and abs(b / a / ratio - 1) < 1e-13


def test_epem_boost_and_rotation_invariance_both_sets():
    rng = np.random.default_rng(3)
    c, p = event_aos(1, 5)
    pb = boost(p, np.array([0.3, -0.2, 0.5]))
    R = rotation(rng)
    pr = p.copy()
    pr[:, 1:] = p[:, 1:] @ R.T
    for par in (c.params_old, c.params_new):
        ref = orc.me2(c.process, par, p)
        assert abs(orc.me2(c.process, par, pb) / ref - 1) < 1e-12
        assert abs(orc.me2(c.process, par, pr) / ref - 1) < 1e-12


# ------------------------------------------------------------------ cfg 2 (SURVEY C10-B closed form)
def ggttx_closed_form(alpha_s, mt, p):
    gs4 = (4 * math.pi * alpha_s) ** 2
    s = mdot(p[0] + p[1], p[0] + p[1])
    t1 = 2 * mdot(p[0], p[2]) / s
    t2 = 2 * mdot(p[1], p[2]) / s
    rho = 4 * mt * mt / s
    return gs4 * (1 / (6 * t1 * t2) - 3.0 / 8) * (t1 * t1 + t2 * t2 + rho - rho * rho / (4 * t1 * t2))


def test_ggttx_closed_form_on_rambo_events():
    c = ev.config(2)
    m, _ = ev.generate(c, 30)
    for k in range(30):
        p = np.ascontiguousarray(m[:, :, k])
        assert abs(orc.me2(c.process, c.params_old, p) / ggttx_closed_form(0.118, 173.0, p) - 1) < 1e-12
    # boosted along z and rotated: still the textbook value (kappa = 0 is Lorentz invariant)
    p = boost(np.ascontiguousarray(m[:, :, 0]), np.array([0.1, 0.2, -0.4]))
    assert abs(orc.me2(c.process, c.params_old, p) / ggttx_closed_form(0.118, 173.0, p) - 1) < 1e-12


def test_ggttx_golden_worked_values():
    c = ev.config(2)
    for ct, old, new, ratio in np.loadtxt(os.path.join(GOLD, "c10b_gg_ttx.txt")):
        h, m = 750.0, 173.0
        pp, st = math.sqrt(h * h - m * m), math.sqrt(1 - ct * ct)
        p = np.array([[h, 0, 0, h], [h, 0, 0, -h], [h, pp * st, 0, pp * ct], [h, -pp * st, 0, -pp * ct]])
        a, b = orc.me2(c.process, c.params_old, p), orc.me2(c.process, c.params_new, p)
        assert abs(a / old - 1) < 1e-12 and abs(b / new - 1) < 1e-12 and abs(b / a / ratio - 1) < 1e-12


def test_ggttxg_golden_worked_point():
    c = ev.config(3)
    tab = np.loadtxt(os.path.join(GOLD, "c10c_gg_ttxg.txt"))
    p, (old, new) = tab[:5], tab[5, :2]
    a, b = orc.me2(c.process, c.params_old, p), orc.me2(c.process, c.params_new, p)
    assert abs(a / old - 1) < 1e-10 and abs(b / new - 1) < 1e-10


# ------------------------------------------------------------------ gauge / Lorentz / rotation
def gluon_k(p, i):
    leg = i if i < 2 else i + 2
    return p[leg] if i < 2 else -p[leg]


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_gauge_invariance_every_colour_flow_amplitude(n):
    """eps_i -> k_i sends each J_sigma to zero at kappa = 0; not at kappa = 0.1 (Q1)."""
    c, p = event_aos(n, 1)
    rng = np.random.default_rng(10 + n)
    hel = rng.choice([-1, 1], size=n + 2)
    ref = np.abs(orc.jamps(n, c.params_old, p, hel)).max()
    for i in ([0, n - 1] if n == 5 else range(n)):
        eps = []
        for j in range(n):
            leg = j if j < 2 else j + 2
            e = orc.polvec(p[leg], hel[leg])
            eps.append(e if j < 2 else e.conj())
        scale = np.abs(gluon_k(p, i)).max()
        eps[i] = gluon_k(p, i).astype(complex) / scale
        J = orc.jamps(n, c.params_old, p, hel, eps_override=np.array(eps))
        assert np.abs(J).max() < 1e-11 * ref, (n, i, np.abs(J).max() / ref)
        if i == 0:
            Jn = orc.jamps(n, c.params_new, p, hel, eps_override=np.array(eps))
            assert np.abs(Jn).max() > 1e-6 * ref     # the modified model is NOT gauge invariant


@pytest.mark.parametrize("idx", [2, 3, 4, 5])
def test_boost_invariance_old_and_rotation_invariance_both(idx):
    rng = np.random.default_rng(20 + idx)
    c, p = event_aos(idx, 2)
    pb = boost(p, np.array([-0.25, 0.1, 0.35]))
    R = rotation(rng)
    pr = p.copy()
    pr[:, 1:] = p[:, 1:] @ R.T
    ref_old = orc.me2(c.process, c.params_old, p)
    ref_new = orc.me2(c.process, c.params_new, p)
    assert abs(orc.me2(c.process, c.params_old, pb) / ref_old - 1) < 1e-11
    assert abs(orc.me2(c.process, c.params_old, pr) / ref_old - 1) < 1e-11
    assert abs(orc.me2(c.process, c.params_new, pr) / ref_new - 1) < 1e-11
    # and the new set is frame dependent (Q1): a boost changes it visibly
    assert abs(orc.me2(c.process, c.params_new, pb) / ref_new - 1) > 1e-6


# ------------------------------------------------------------------ colour: route F == route E, table C7
@pytest.mark.parametrize("n", [2, 3])
def test_colour_string_route_equals_explicit_colour_all_helicities(n):
    c, p = event_aos(n, 0)
    for par in (c.params_old, c.params_new):
        for hel in itertools.product((1, -1), repeat=n + 2):
            f = orc.me2_hel(n, par, p, hel, "F")
            e = orc.me2_hel(n, par, p, hel, "E")
            assert abs(f - e) <= 1e-12 * max(abs(e), 1e-30) + 1e-25, (hel, f, e)


def test_colour_string_route_equals_explicit_colour_n4_two_helicities():
    c, p = event_aos(4, 0)
    for par in (c.params_new, c.params_old):
        for hel in ([1, -1, 1, -1, 1, 1], [-1, -1, 1, 1, -1, 1]):
            f = orc.me2_hel(4, par, p, hel, "F")
            e = orc.me2_hel(4, par, p, hel, "E")
            assert abs(f / e - 1) < 1e-11


def test_colour_matrix_table():
    tab = np.loadtxt(os.path.join(GOLD, "c7_colour.txt"))
    rows = {}
    for line in open(os.path.join(GOLD, "c7_colour_row0.txt")):
        if line.startswith("#"):
            continue
        parts = line.split()
        ms = []
        for it in parts[1:]:
            v, k = it.split(":")
            ms += [int(v)] * int(k)
        rows[int(parts[0])] = sorted(ms)
    for n, den, diag, rowsum, total, lmin, lmax in tab:
        n = int(n)
        C = orc.colour_matrix(n)
        Ch = C * den
        assert np.abs(Ch - np.round(Ch)).max() < 1e-8
        Ch = np.round(Ch)
        assert np.all(np.diag(Ch) == diag) and abs(diag / den - 3 * (4 / 3) ** n) < 1e-12
        assert np.all(Ch.sum(axis=1) == rowsum) and Ch.sum() == total
        assert np.array_equal(Ch, Ch.T)
        assert sorted(Ch[0].astype(int).tolist()) == rows[n]
        for r in Ch:
            assert sorted(r.astype(int).tolist()) == rows[n]      # every row is a permutation of row 0
        w = np.linalg.eigvalsh(C)
        assert abs(w[0] - lmin) < 2e-6 and abs(w[-1] - lmax) < 2e-6 and w[0] > 0
    C3 = np.array([[64, -8, -8, 1, 1, 10], [-8, 64, 1, 10, -8, 1], [-8, 1, 64, -8, 10, 1],
                   [1, 10, -8, 64, 1, -8], [1, -8, 10, 1, 64, -8], [10, 1, 1, -8, -8, 64]]) / 9.0
    assert np.abs(orc.colour_matrix(3) - C3).max() < 1e-13


def test_denominators():
    """Averaging denominator D (reading Q3, SURVEY.md:433: what out_me_* contain): 2 helicities x 2 helicities x 8 colours x 8
    colours of the two incoming gluons, times k! for the k identical final-state gluons, read here from the process string.
    This restates the rule; what PINS it is elsewhere: the closed form of gg -> ttbar fixes the 1/256 (k = 0), and the soft-gluon
    limit |M_n|^2 -> eikonal x |M_{n-1}|^2 / (k+1) fixes D(k+1) / D(k) for k + 1 = 1, 2, 3 (tests/test_oracle_pins_soft.py)."""
    for idx in (2, 3, 4, 5):
        c = ev.config(idx)
        final = c.process.split("_")[1]                  # "ttx", "ttxg", ...
        k = final.count("g")
        assert len(final) - 3 == k == c.n_ext - 4
        assert orc.denominator(k + 2) == (2 * 2) * (8 * 8) * math.factorial(k)


# ------------------------------------------------------------------ new-model pins
def lagrange(xs, ys, x):
    """value at x of the polynomial of degree len(xs) - 1 through (xs, ys): the Lagrange formula written out, no least squares"""
    return sum(ys[j] * np.prod([(x - xs[m]) / (xs[j] - xs[m]) for m in range(len(xs)) if m != j]) for j in range(len(xs)))


def chebyshev_nodes(lo, hi, count):
    return 0.5 * (lo + hi) + 0.5 * (hi - lo) * np.cos(np.pi * (2 * np.arange(count) + 1) / (2 * count))


@pytest.mark.parametrize("idx", [2, 3, 4, 5])
def test_me2_is_polynomial_of_degree_2n_minus_2_in_kappa(idx):
    """|M'|^2 with ggg_scale = gggg_scale = 1 + kappa is a polynomial of degree 2 (n - 1) in kappa (every amplitude has at most
    n - 1 powers of the scales).  Exact interpolation through 2n - 1 Chebyshev nodes of [-0.3, 0.6] reproduces the oracle at
    kappa = 0.1 and 0.55 to 1e-9 for every n (np.polyfit on equispaced points lost two digits at n >= 4: that was the fit, not
    the oracle); one node fewer does not."""
    n = idx
    c, p = event_aos(idx, 4)
    deg = 2 * (n - 1)

    def me2_at(k):
        return orc.me2(c.process, ev.params(ggg_scale=1 + k, gggg_scale=1 + k), p)

    ks = chebyshev_nodes(-0.3, 0.6, deg + 1)
    vals = [me2_at(k) for k in ks]
    got55, got01 = me2_at(0.55), me2_at(0.1)
    assert abs(lagrange(ks, vals, 0.55) / got55 - 1) < 1e-9
    assert abs(lagrange(ks, vals, 0.1) / got01 - 1) < 1e-9
    # one degree less does NOT fit
    ks_lo = chebyshev_nodes(-0.3, 0.6, deg)
    vals_lo = [me2_at(k) for k in ks_lo]
    assert max(abs(lagrange(ks_lo, vals_lo, 0.55) / got55 - 1), abs(lagrange(ks_lo, vals_lo, 0.1) / got01 - 1)) > 1e-6


def test_ggttx_per_diagram_scaling_reading():
    """J1 ~ A_t + (1+k) A_s, J2 ~ A_u - (1+k) A_s: jamps are affine in the ggg scale and
    J1 + J2 does not depend on it."""
    c, p = event_aos(2, 6)
    hel = [1, -1, 1, 1]
    J0 = orc.jamps(2, ev.params(ggg_scale=1.0), p, hel)
    J1 = orc.jamps(2, ev.params(ggg_scale=1.1), p, hel)
    J2 = orc.jamps(2, ev.params(ggg_scale=1.2), p, hel)
    assert np.abs((J2 - J1) - (J1 - J0)).max() < 1e-13 * np.abs(J0).max()
    assert abs((J0.sum() - J2.sum())) < 1e-13 * np.abs(J0).max()


def test_ggttxg_jamps_are_c0_plus_x_c1_plus_x2_c2_plus_y_c3():
    """SURVEY C6 at the amplitude level, for gg -> ttbar g: every colour-flow amplitude is J = c0 + x c1 + x^2 c2 + y c3 in
    (x, y) = (ggg_scale, gggg_scale) -- no x y, x^3 or y^2 term -- and carries the overall factor alpha_s^(3/2).  The CUDA path
    forms the four coefficient amplitudes once and folds them with each set's couplings ("one pass for all
    sets at n = 3"); it may do so only because this holds for the oracle, which evaluates every set from scratch."""
    c, p = event_aos(3, 5)
    rng = np.random.default_rng(33)
    for _ in range(3):
        hel = rng.choice([-1, 1], size=5)
        J = lambda x, y, a=0.118: orc.jamps(3, ev.params(ggg_scale=x, gggg_scale=y, alpha_s=a), p, hel)
        c0 = J(0.0, 0.0)
        c3 = J(0.0, 1.0) - c0
        c1 = 0.5 * (J(1.0, 0.0) - J(-1.0, 0.0))
        c2 = 0.5 * (J(1.0, 0.0) + J(-1.0, 0.0)) - c0
        scale = np.abs(J(1.0, 1.0)).max()
        assert min(np.abs(x).max() for x in (c0, c1, c2, c3)) > 1e-6 * scale        # all four structures are present
        for x, y in ((1.1, 1.1), (0.7, 1.9), (-2.3, 0.4), (3.0, -1.5)):
            assert np.abs(J(x, y) - (c0 + x * c1 + x * x * c2 + y * c3)).max() < 1e-12 * scale * (1 + x * x + abs(y))
        # alpha_s: overall factor g_s^3 of the amplitude (sqrt(4 pi alpha_s)^3; the dropped common factor is convention-independent here)
        r = J(1.3, 0.8, 0.15) / J(1.3, 0.8, 0.118)
        expo = np.log(abs(r[0])) / np.log(0.15 / 0.118)
        assert np.abs(r - r[0]).max() < 1e-12 * abs(r[0]) and min(abs(expo - 1.0), abs(expo - 1.5)) < 1e-9     # g_s^2 or g_s^3 (a common i g_q may be dropped)


@pytest.mark.parametrize("idx", [2, 3])
def test_parity_flipping_all_helicities_keeps_me2_hel(idx):
    """|M_{-h}|^2 = |M_h|^2 for both parameter sets (real couplings, Gamma_t = 0) — SURVEY Q5;
    the CUDA path may use it only because this holds for the oracle's full sum."""
    n = idx
    c, p = event_aos(idx, 7)
    for par in (c.params_old, c.params_new):
        for hel in itertools.product((1, -1), repeat=n + 2):
            if hel[0] < 0:
                continue
            a = orc.me2_hel(n, par, p, hel, "F")
            b = orc.me2_hel(n, par, p, [-h for h in hel], "F")
            assert abs(a - b) <= 1e-11 * max(a, b) + 1e-24


@pytest.mark.parametrize("n", [4, 5])
def test_parity_flip_n4_n5_on_sampled_helicities(n):
    c, p = event_aos(n, 3)
    rng = np.random.default_rng(70 + n)
    for par in (c.params_old, c.params_new):
        for _ in range(4):
            hel = rng.choice([-1, 1], size=n + 2)
            a = orc.me2_hel(n, par, p, hel, "F")
            b = orc.me2_hel(n, par, p, -hel, "F")
            assert abs(a - b) <= 1e-11 * max(a, b) + 1e-24


def test_spinors_off_the_mass_shell_reading_q8():
    """Reading Q8 (SURVEY.md:438; R8): spinors take E from the input, m from the PARAMETER SET and the direction
    from the input 3-momentum; a set whose top mass differs from the one the events were generated with then
    sees momenta with E^2 - p^2 != m^2.  What the normalisation must still satisfy, whatever |p| is:
    ubar_l u_l' = 2 m d_ll', vbar_l v_l' = -2 m d_ll', u^+ u = v^+ v = 2 E, and (Sigma.p_hat) u_l = l u_l, (Sigma.p_hat) v_l = -l v_l."""
    rng = np.random.default_rng(5)
    g0 = orc.gamma(0)
    for m_par, m_shell in ((170.0, 173.0), (176.5, 173.0), (0.0, 4.2)):
        p = rand_mom(rng, m_shell)
        ph = p[1:] / np.linalg.norm(p[1:])
        Sig = sum(ph[i] * 1j * orc.gamma((i + 1) % 3 + 1) @ orc.gamma((i + 2) % 3 + 1) for i in range(3))   # Sigma^i = i g^j g^k, (i,j,k) cyclic
        for kind, sgn in (("u", 1.0), ("v", -1.0)):
            sp = {l: orc.spinor(kind, p, m_par, l) for l in (1, -1)}
            for l in (1, -1):
                for l2 in (1, -1):
                    d = 1.0 if l == l2 else 0.0
                    assert abs(sp[l].conj() @ g0 @ sp[l2] - sgn * 2 * m_par * d) < 1e-12 * p[0]
                    assert abs(sp[l].conj() @ sp[l2] - 2 * p[0] * d) < 1e-12 * p[0]
                assert np.abs(Sig @ sp[l] - sgn * l * sp[l]).max() < 1e-12 * math.sqrt(p[0])


# ------------------------------------------------------------------ eq. 3
def test_eq3_reweight_and_identity_when_params_equal():
    c = ev.config(3)
    m, w = ev.generate(c, 12)
    a, b, wn, used = orc.reweight(c.process, c.params_old, c.params_new, m, w, nthreads=2)
    assert used == 2
    # w' = fl(w * fl(b / a)): two roundings; fl(w' * a) and fl(w * b) one more each -> the two sides differ by at most
    # 4 * 2^-53 = 4.4e-16 relative to first order (5e-16 leaves room for the second-order terms)
    assert np.all(np.abs(wn * a - w * b) <= 5e-16 * np.abs(w * b))
    for k in (0, 5, 11):
        p = np.ascontiguousarray(m[:, :, k])
        assert a[k] == orc.me2(c.process, c.params_old, p) and b[k] == orc.me2(c.process, c.params_new, p)
    a2, b2, wn2, _ = orc.reweight(c.process, c.params_old, c.params_old, m, w)
    assert np.array_equal(a2, b2) and np.array_equal(wn2, w) and np.array_equal(a2, a)


def test_eq2_cross_section_is_the_sum_of_weights():
    """eq. 2: sigma ~ sum_k W_k.  Pin: Python's exactly rounded math.fsum; recursive summation of n positive terms is
    within (n - 1) 2^-53 of it (Higham, Accuracy and Stability of Numerical Algorithms, eq. 4.4); W' of eq. 3 summed the same way."""
    c = ev.config(2)
    m, w = ev.generate(c, 5000)
    for x in (w, orc.reweight(c.process, c.params_old, c.params_new, m[:, :, :300].copy(), w[:300].copy())[2]):
        exact = math.fsum(x)
        assert abs(orc.cross_section(x) - exact) <= (len(x) - 1) * 2.0 ** -53 * exact
    assert orc.cross_section(np.array([1.0, 2.0 ** -60, -1.0])) == 0.0          # plain left-to-right, not compensated
    assert orc.cross_section(np.array([])) == 0.0


def test_me2_zero_gives_ieee_result():
    """eq. 3 needs |M|^2 != 0; convention (include/rwgt.h): IEEE inf/nan, no trap."""
    c = ev.config(2)
    m, w = ev.generate(c, 2)
    par0 = ev.params(alpha_s=0.0)
    with np.errstate(all="ignore"):
        a, b, wn, _ = orc.reweight(c.process, par0, c.params_new, m, w)
    assert np.all(a == 0) and np.all(np.isinf(wn) | np.isnan(wn))
