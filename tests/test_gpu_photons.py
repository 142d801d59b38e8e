"""GPU parity of e+ e- -> n photons (n = 5: the process the paper measured) against the CPU oracle,
through the C ABI.  FP64, 1e-11 relative per event for each of |M|^2, |M'|^2, W' (north_star tolerance)."""
import numpy as np
import pytest

import oracle as orc
from paper_2312_07440_b200 import binding as B, events as ev
from test_gpu_parity import gpu_run, rel, TOL64

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

# several 16-event groups plus a ragged tail; the n = 5 oracle costs ~0.1 s per event and parameter set
SIZES = {2: 5003, 3: 2051, 4: 515, 5: 83}


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_fp64_parity_every_event(n):
    c = ev.photon_config(n)
    m, w = ev.generate(c, SIZES[n])
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, m, w)
    got = gpu_run(c.process, c.params_old, c.params_new, m, w)
    for g, ref, name in zip(got, (a, b, wn), ("me_old", "me_new", "w_new")):
        e = rel(g, ref)
        assert e.max() < TOL64, (c.process, name, int(e.argmax()), e.max())


def test_full_size_bench_launch_sampled_against_oracle():
    c = ev.config(6)
    m, w = ev.generate(c)
    got = gpu_run(c.process, c.params_old, c.params_new, m, w)
    assert np.all(np.isfinite(got)) and np.all(got[0] > 0)
    idx = np.unique(np.concatenate([[0, 15, 16, c.n_events - 17, c.n_events - 1], np.random.default_rng(6).integers(0, c.n_events, 24)]))
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, np.ascontiguousarray(m[:, :, idx]), w[idx])
    for g, ref in zip(got[:, idx], (a, b, wn)):
        assert rel(g, ref).max() < TOL64
    # property at any size: the weight ratio of every event is (alpha'/alpha)^5
    r = (c.params_new[0] / c.params_old[0]) ** 5
    assert np.abs(got[1] / got[0] / r - 1).max() < 1e-14 and np.abs(got[2] / (w * r) - 1).max() < 1e-14


def test_identical_parameter_sets_give_ratio_exactly_one():
    c = ev.photon_config(5)
    m, w = ev.generate(c, 333)
    got = gpu_run(c.process, c.params_old, c.params_old, m, w)
    assert np.array_equal(got[0], got[1]) and np.array_equal(got[2], w)


def test_multi_set_random_couplings_and_host_path():
    # the paper's use: a new electroweak coupling per reweight iteration, K sets in one pass (PAPER.md:87 step 7)
    c = ev.photon_config(5)
    m, w = ev.generate(c, 70001)
    rng = np.random.default_rng(77)
    sets = [ev.params(alpha_em=float(x)) for x in rng.uniform(0.5, 2.0, size=6) / 132.5]
    K = len(sets)
    r = B.Reweighter(c.process, c.params_old, sets, "fp64")
    got = r.run(torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda())
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    r.close()
    me_old, me_new, w_new = got[0], got[1:1 + K], got[1 + K:]
    sample = np.arange(0, 70001, 7001)
    for k, s in enumerate(sets):
        a, b, wn, _ = orc.reweight(c.process, c.params_old, s, np.ascontiguousarray(m[:, :, sample]), w[sample])
        assert rel(me_old[sample], a).max() < TOL64 and rel(me_new[k][sample], b).max() < TOL64 and rel(w_new[k][sample], wn).max() < TOL64
        assert np.abs(w_new[k] / (w * (s[0] / c.params_old[0]) ** 5) - 1).max() < 1e-14
    h = B.rwgt_create_multi(c.process, c.params_old, sets)
    h_old, h_new, h_w = np.empty(70001), np.empty((K, 70001)), np.empty((K, 70001))
    B.rwgt_run_multi_host(h, m, w, h_old, h_new, h_w)
    B.rwgt_destroy(h)
    assert np.array_equal(h_old, me_old) and np.array_equal(h_new, me_new) and np.array_equal(h_w, w_new)


def test_rotation_invariance_on_gpu():
    c = ev.photon_config(5)
    m, w = ev.generate(c, 257)
    q, rr = np.linalg.qr(np.random.default_rng(2).normal(size=(3, 3)))
    q = q @ np.diag(np.sign(np.diag(rr)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    m2 = m.copy()
    m2[:, 1:, :] = np.einsum("ij,pjn->pin", q, m[:, 1:, :])
    g1 = gpu_run(c.process, c.params_old, c.params_new, m, w)
    g2 = gpu_run(c.process, c.params_old, c.params_new, m2, w)
    assert rel(g2[0], g1[0]).max() < 1e-10


def test_bad_arguments():
    c = ev.photon_config(5)
    with pytest.raises(Exception):
        B.Reweighter("epem_aaaaaa", c.params_old, c.params_new)
    with pytest.raises(Exception):
        B.Reweighter(c.process, c.params_old, c.params_new, "fp32")      # FP64 only
