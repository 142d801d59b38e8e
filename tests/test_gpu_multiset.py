"""GPU parity of the K-parameter-set pass (PAPER.md:87 step 7): rwgt_create_multi /
rwgt_run_multi against the CPU oracle evaluated once per set, element by element."""
import numpy as np
import pytest

import oracle as orc
from paper_2312_07440_b200 import binding as B, events as ev

pytestmark = pytest.mark.gpu
TOL64 = 1e-11
torch = pytest.importorskip("torch")


def rel(got, ref):
    return np.abs(got / ref - 1)


def new_sets(idx):
    c = ev.config(idx)
    if idx == 1:
        return [c.params_new, ev.params(GammaZ=2.3, sin2_thetaW=0.2250), ev.params(mZ=92.5, alpha_em=1 / 128.0), c.params_old.copy()]
    return [c.params_new, ev.params(ggg_scale=0.9, gggg_scale=0.8), ev.params(ggg_scale=1.25, gggg_scale=1.1, alpha_s=0.13),
            c.params_old.copy(), ev.params(ggg_scale=-1.0, gggg_scale=1.0)]


def run_multi(c, sets, m, w, precision="fp64"):
    r = B.Reweighter(c.process, c.params_old, sets, precision)
    out = r.run(torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda())
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    r.close()
    return res


@pytest.mark.parametrize("idx,n", [(1, 3001), (2, 2049), (3, 601), (4, 103), (5, 19)])
def test_multi_set_fp64_parity_every_event(idx, n):
    c = ev.config(idx)
    sets = new_sets(idx)
    K = len(sets)
    m, w = ev.generate(c, n)
    got = run_multi(c, sets, m, w)
    assert got.shape == (1 + 2 * K, n)
    for k, pn in enumerate(sets):
        a, b, wn, _ = orc.reweight(c.process, c.params_old, pn, m, w)
        for g, ref, name in ((got[0], a, "me_old"), (got[1 + k], b, "me_new"), (got[1 + K + k], wn, "w_new")):
            e = rel(g, ref)
            assert e.max() < TOL64, (c.process, k, name, int(e.argmax()), e.max())
    # the set equal to the old one: ratio exactly 1 (north_star), bitwise
    k_same = 3
    assert np.array_equal(got[1 + k_same], got[0]) and np.array_equal(got[1 + K + k_same], w)


@pytest.mark.parametrize("idx,n", [(2, 515), (3, 301), (4, 47), (5, 7)])
def test_multi_set_with_different_top_masses(idx, n):
    """Sets with other top masses make the library redo externals, momentum sums and denominators for those sets (R12).
    The events stay on the old set's mass shell; off shell both sides normalise the spinors from (E, m_t') (reading Q8 / R8)."""
    c = ev.config(idx)
    sets = [ev.params(mt=170.0, ggg_scale=1.1, gggg_scale=1.1), c.params_new, ev.params(mt=178.25, ggg_scale=0.7), ev.params(mt=173.0, alpha_s=0.11)]
    m, w = ev.generate(c, n)
    got = run_multi(c, sets, m, w)
    K = len(sets)
    for k, pn in enumerate(sets):
        a, b, wn, _ = orc.reweight(c.process, c.params_old, pn, m, w)
        assert rel(got[0], a).max() < TOL64 and rel(got[1 + k], b).max() < TOL64 and rel(got[1 + K + k], wn).max() < TOL64


def test_multi_set_matches_single_set_calls_bitwise_and_max_sets():
    """K sets in one pass (evaluated set by set: four generic sets of n = 4 have rank 5, no saving) give bit-identical numbers to K
    separate (old, new_k) handles; K = RWGT_MAX_SETS works, K = RWGT_MAX_SETS + 1 is refused."""
    c = ev.config(4)
    sets = [ev.params(ggg_scale=1.1, gggg_scale=0.9), ev.params(ggg_scale=0.8, gggg_scale=1.3), ev.params(ggg_scale=1.4, gggg_scale=1.05),
            ev.params(ggg_scale=0.6, gggg_scale=0.7)]
    m, w = ev.generate(c, 57)
    got = run_multi(c, sets, m, w)
    K = len(sets)
    dm, dw = torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda()
    for k in range(K):
        r = B.Reweighter(c.process, c.params_old, sets[k])
        one = r.run(dm, dw).cpu().numpy()
        r.close()
        assert np.array_equal(one[0], got[0]) and np.array_equal(one[1], got[1 + k]) and np.array_equal(one[2], got[1 + K + k])
    many = [ev.params(ggg_scale=1 + k, gggg_scale=1 + k) for k in np.linspace(-0.3, 0.45, B.RWGT_MAX_SETS)]
    assert run_multi(c, many, m, w).shape == (1 + 2 * B.RWGT_MAX_SETS, 57)
    with pytest.raises(RuntimeError, match="RWGT_MAX_SETS"):
        B.rwgt_create_multi(c.process, c.params_old, many + [many[0]])
    h = B.rwgt_create_multi(c.process, c.params_old, sets[:3])
    assert B.rwgt_n_sets(h) == 3
    with pytest.raises(RuntimeError, match="rwgt_run_multi"):
        B.rwgt_run(h, 1, 1, 1, 1, 1, 5)              # single-set entry point refuses a multi-set handle
    B.rwgt_destroy(h)


def poly_sets(kind, K):
    if kind == "diagonal":         # the bench's Fig. 3 axis: ggg = gggg = 1 + kappa_k
        return [ev.params(ggg_scale=1 + 0.1 * (k + 1) / K, gggg_scale=1 + 0.1 * (k + 1) / K) for k in range(K)]
    rng = np.random.default_rng(K)
    if kind == "general":          # both scales independent, alpha_s too
        return [ev.params(ggg_scale=float(x), gggg_scale=float(y), alpha_s=float(a)) for x, y, a in
                zip(rng.uniform(0.7, 1.3, K), rng.uniform(0.7, 1.3, K), rng.uniform(0.10, 0.13, K))]
    return [ev.params(ggg_scale=float(x), alpha_s=float(a)) for x, a in zip(rng.uniform(0.5, 1.5, K), rng.uniform(0.10, 0.13, K))]   # ggg only


@pytest.mark.parametrize("idx,n,kind,K,precision", [(4, 41, "diagonal", 15, "fp64"), (4, 23, "general", 12, "fp64"), (4, 23, "ggg", 9, "fp64"),
                                                    (5, 5, "diagonal", 15, "fp64"), (5, 3, "ggg", 7, "fp64"), (4, 41, "diagonal", 15, "fp32"),
                                                    (5, 5, "diagonal", 15, "mixed")])
def test_coupling_only_sets_polynomial_mode_against_oracle(idx, n, kind, K, precision):
    """sets that differ only in ggg_scale / gggg_scale / alpha_s are exact linear combinations of a few node sets (the
    amplitudes are polynomials in the two scales); every set against the oracle's own full evaluation of that set; a set
    equal to the old one gives W' = W bitwise (same weights, same factor)."""
    c = ev.config(idx)
    sets = poly_sets(kind, K)
    sets.insert(3, c.params_old.copy())
    K += 1
    m, w = ev.generate(c, n)
    got = run_multi(c, sets, m, w, precision)
    tmax, tmed = (TOL64, TOL64) if precision == "fp64" else (1e-4, 1e-6 if n > 20 else 1e-5)
    for k, pn in enumerate(sets):
        a, b, wn, _ = orc.reweight(c.process, c.params_old, pn, m, w)
        for g, ref in ((got[0], a), (got[1 + k], b), (got[1 + K + k], wn)):
            e = rel(g, ref)
            assert e.max() < tmax and np.median(e) < tmed, (kind, k, e.max(), np.median(e))
    assert np.array_equal(got[1 + 3], got[0]) and np.array_equal(got[1 + K + 3], w)


def test_polynomial_mode_is_deterministic_and_costs_less_than_a_loop():
    """rwgt_flops_per_event reflects the mode: 16 diagonal sets of n = 5 need five node evaluations (degree n - 1 in kappa), not 17."""
    c = ev.config(5)
    h1 = B.rwgt_create(c.process, c.params_old, c.params_new)
    h16 = B.rwgt_create_multi(c.process, c.params_old, poly_sets("diagonal", 16))
    f1, f16 = B.rwgt_flops_per_event(h1), B.rwgt_flops_per_event(h16)
    assert 2.3 < f16 / f1 < 2.7                      # 5 evaluations against 2
    B.rwgt_destroy(h1)
    B.rwgt_destroy(h16)
    m, w = ev.generate(c, 301)
    r = B.Reweighter(c.process, c.params_old, poly_sets("diagonal", 16))
    dm, dw = torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda()
    ref = r.run(dm, dw).clone()
    for _ in range(3):
        assert torch.equal(r.run(dm, dw), ref)
    r.close()


@pytest.mark.parametrize("precision", ["fp32", "mixed"])
def test_multi_set_fp32_and_mixed(precision):
    c = ev.config(4)
    sets = new_sets(4)[:3]
    m, w = ev.generate(c, 203)
    got = run_multi(c, sets, m, w, precision)
    K = len(sets)
    for k, pn in enumerate(sets):
        a, b, wn, _ = orc.reweight(c.process, c.params_old, pn, m, w)
        for g, ref in ((got[0], a), (got[1 + k], b), (got[1 + K + k], wn)):
            e = rel(g, ref)
            assert e.max() < 1e-4 and np.median(e) < 1e-6, (precision, k, e.max(), np.median(e))


def test_multi_set_host_path_chunked():
    c = ev.config(2)
    sets = new_sets(2)[:3]
    n = 2 * 65536 + 11
    m0, w0 = ev.generate(c, 2048)
    reps = (n + 2047) // 2048
    m, w = np.tile(m0, (1, 1, reps))[:, :, :n].copy(), np.tile(w0, reps)[:n].copy()
    dev = run_multi(c, sets, m, w)
    h = B.rwgt_create_multi(c.process, c.params_old, sets)
    a, b, o = np.empty(n), np.empty((3, n)), np.empty((3, n))
    B.rwgt_run_multi_host(h, m, w, a, b, o)
    B.rwgt_destroy(h)
    assert np.array_equal(a, dev[0]) and np.array_equal(b, dev[1:4]) and np.array_equal(o, dev[4:7])


@pytest.mark.parametrize("K", [1, 2, 3, 4, 16])
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_gg_ttxg_one_pass_for_all_sets_odd_and_even_counts(K, precision):
    """gg -> ttbar g evaluates the currents once for all sets of equal mass and folds the coefficient amplitudes two sets at a time
    (QuarkLine3F): odd and even totals (the last chunk of an odd total holds one set), couplings that differ in
    alpha_s, ggg and gggg scale separately, against the oracle per set; a set equal to the old one reproduces W bitwise."""
    c = ev.config(3)
    rng = np.random.default_rng(300 + K)
    sets = [ev.params(ggg_scale=float(1 + rng.uniform(-0.4, 0.4)), gggg_scale=float(1 + rng.uniform(-0.4, 0.4)), alpha_s=float(rng.uniform(0.09, 0.14)))
            for _ in range(K)]
    sets[K // 2] = c.params_old.copy()
    n = 413
    m, w = ev.generate(c, n)
    got = run_multi(c, sets, m, w, precision)
    tol = TOL64 if precision == "fp64" else 1e-4
    for k, pn in enumerate(sets):
        a, b, wn, _ = orc.reweight(c.process, c.params_old, pn, m, w)
        assert rel(got[0], a).max() < tol and rel(got[1 + k], b).max() < tol and rel(got[1 + K + k], wn).max() < tol, (K, k)
    assert np.array_equal(got[1 + K // 2], got[0]) and np.array_equal(got[1 + K + K // 2], w)
