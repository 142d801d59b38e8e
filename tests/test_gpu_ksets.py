"""GPU parity of the K-set pass AT THE SIZES bench.py TIMES IT (PAPER.md:87 step 7 "Repeat steps 4 - 6 for all parameter sets";
PAPER.md:117 Fig. 3; SURVEY.md:531-532 D3).

bg_kernel is persistent (one CTA per SM, event groups handed out round after round), so its group loop, the amplitude-buffer
hand-over between groups and the reuse of the polynomial mode's scratch only run when a launch holds more than 148 x (events in
flight per CTA) events.  The tests of test_gpu_multiset.py stay below that.  Here the FULL seeded event set of cfgs 3-5 is launched
with each named list of new parameter sets (events.kset_list: the lists bench.py times, independent coupling scales, other top
masses) in FP64, FP32 and mixed precision and compared, per set and element by element, with oracle values stored by
tests/golden/make_goldens.py --sets on events.kset_sample: a prefix longer than two rounds, a strided sample over every later round,
and the ragged tail.  |M|^2 of the old set is compared on EVERY event (tests/golden/full_cfg<N>.npz), and a set equal to the old one
must give W' = W bitwise over the whole launch.  No oracle time is spent on the GPU box."""
import os

import numpy as np
import pytest

from paper_2312_07440_b200 import binding as B, events as ev

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
GOLD = os.path.join(os.path.dirname(__file__), "golden")
TOL = {"fp64": (1e-11, 1e-11), "fp32": (1e-4, 1e-6), "mixed": (1e-4, 1e-6)}     # (max, median) of the relative error, north_star

CASES = [(i, name, prec) for i, names in ev.KSET_GOLDENS.items() for name in names for prec in ("fp64", "fp32", "mixed")]


def kset_golden(idx, name):
    f = os.path.join(GOLD, f"ksets_cfg{idx}_{name}.npz")
    if not os.path.exists(f):
        pytest.fail(f"{f} missing: run tests/golden/make_goldens.py --config {idx} --sets {name}")
    g = np.load(f)
    c = ev.config(idx)
    sets = ev.kset_list(c, name)
    assert int(g["seed"]) == c.seed and np.array_equal(g["params_old"], c.params_old) and np.array_equal(g["sets"], np.array(sets))
    assert np.array_equal(g["idx"], ev.kset_sample(c))
    return c, sets, g


_events = {}


def full_set(c):
    """the config's full seeded event set on the device (kept across the cases of one config)"""
    if c.index not in _events:
        _events.clear()
        m, w = ev.generate(c)
        _events[c.index] = (w, torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda())
    return _events[c.index]


@pytest.mark.parametrize("idx,name,precision", CASES)
def test_full_size_k_set_launch_against_goldens(idx, name, precision):
    c, sets, g = kset_golden(idx, name)
    K, sel = len(sets), g["idx"]
    w, dm, dw = full_set(c)
    r = B.Reweighter(c.process, c.params_old, sets, precision)
    out = r.run(dm, dw)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    r.close()
    assert got.shape == (1 + 2 * K, c.n_events) and np.all(np.isfinite(got)) and np.all(got[:1 + K] > 0)
    tmax, tmed = TOL[precision]
    # the old set on every event of the launch
    e = np.abs(got[0] / np.load(os.path.join(GOLD, f"full_cfg{idx}.npz"))["out"][0] - 1)
    assert e.max() < tmax and np.median(e) < tmed, (c.process, name, precision, "me_old", int(e.argmax()), e.max(), np.median(e))
    # every new set on the sampled events
    for k in range(K):
        for gk, ref, what in ((got[1 + k, sel], g["me_new"][k], "me_new"), (got[1 + K + k, sel], g["w_new"][k], "w_new")):
            e = np.abs(gk / ref - 1)
            assert e.max() < tmax, (c.process, name, precision, k, what, int(sel[e.argmax()]), e.max())
            assert np.median(e) < tmed, (c.process, name, precision, k, what, np.median(e))
        # eq. 3 on every event of the launch for this set
        assert np.all(np.abs(got[1 + K + k] * got[0] - w * got[1 + k]) <= 5e-16 * np.abs(w * got[1 + k]))
        if np.array_equal(sets[k], c.params_old):     # old == new: |M'|^2 = |M|^2 and W' = W, bitwise, on every event
            assert np.array_equal(got[1 + k], got[0]) and np.array_equal(got[1 + K + k], w), (c.process, name, precision, k)


@pytest.mark.parametrize("idx", [3, 4, 5])
def test_full_size_k_set_launch_is_repeatable_and_matches_the_single_set_launch(idx):
    """Two launches of one handle give the same bits (nothing left over from a launch, no schedule dependence), and set k of the
    K-set pass agrees with a launch of that set alone within the FP64 tolerance on every event (bitwise outside the polynomial
    mode's interpolation is not required)."""
    c = ev.config(idx)
    name = ev.KSET_GOLDENS[idx][0]
    sets = ev.kset_list(c, name)
    K = len(sets)
    w, dm, dw = full_set(c)
    r = B.Reweighter(c.process, c.params_old, sets)
    a = r.run(dm, dw).cpu().numpy()
    b = r.run(dm, dw).cpu().numpy()
    r.close()
    assert np.array_equal(a, b)
    k = K - 1
    r1 = B.Reweighter(c.process, c.params_old, sets[k])
    one = r1.run(dm, dw).cpu().numpy()
    r1.close()
    assert np.abs(a[0] / one[0] - 1).max() < 1e-11 and np.abs(a[1 + k] / one[1] - 1).max() < 1e-11 and np.abs(a[1 + K + k] / one[2] - 1).max() < 1e-11
