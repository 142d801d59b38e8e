"""GPU parity against the full-set expected values tests/golden/full_cfg<N>.npz (written by tests/golden/make_goldens.py, which
calls only the CPU oracle): FP64, FP32 and mixed launches at BASELINE.json's sizes, in the launch configuration bench.py times,
compared element by element over every stored event; max AND median of the per-event relative error asserted per output
(reading Q9, SURVEY.md:439: both statistics run over all events of the config; D3, SURVEY.md:531-532).
No oracle time is spent on the GPU box."""
import os

import numpy as np
import pytest

from paper_2312_07440_b200 import binding as B, events as ev

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
GOLD = os.path.join(os.path.dirname(__file__), "golden")
TOL = {"fp64": (1e-11, 1e-11), "fp32": (1e-4, 1e-6), "mixed": (1e-4, 1e-6)}
NAMES = ("me_old", "me_new", "w_new")


def golden(idx):
    f = os.path.join(GOLD, f"full_cfg{idx}.npz")
    if not os.path.exists(f):
        pytest.fail(f"{f} missing: run tests/golden/make_goldens.py --config {idx}")
    g = np.load(f)
    c = ev.config(idx)
    assert int(g["seed"]) == c.seed and np.array_equal(g["params_old"], c.params_old) and np.array_equal(g["params_new"], c.params_new)
    return c, g["out"]


CASES = [(1, "fp64"), (2, "fp64"), (3, "fp64"), (3, "fp32"), (3, "mixed"), (4, "fp64"), (4, "fp32"), (4, "mixed"),
         (5, "fp64"), (5, "fp32"), (5, "mixed"), (6, "fp64")]


@pytest.mark.parametrize("idx,precision", CASES)
def test_full_size_launch_against_goldens(idx, precision):
    c, ref = golden(idx)
    ngold = ref.shape[1]
    m, w = ev.generate(c)                          # the launch bench.py times: all n_events of the config
    r = B.Reweighter(c.process, c.params_old, c.params_new, precision)
    out = r.run(torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda())
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    r.close()
    assert np.all(np.isfinite(got)) and np.all(got[:2] > 0)
    tmax, tmed = TOL[precision]
    for k, name in enumerate(NAMES):
        e = np.abs(got[k, :ngold] / ref[k] - 1)
        assert e.max() < tmax, (c.process, precision, name, ngold, int(e.argmax()), e.max())
        assert np.median(e) < tmed, (c.process, precision, name, ngold, np.median(e))
    # eq. 3 on every event of the full launch, beyond the stored prefix too
    assert np.all(np.abs(got[2] * got[0] - w * got[1]) <= 5e-16 * np.abs(w * got[1]))


def test_goldens_cover_every_event_of_every_config():
    """parity on every event of each config at least once."""
    for idx in (1, 2, 3, 4, 5, 6):
        c, ref = golden(idx)
        assert ref.shape[1] == c.n_events and np.all(np.isfinite(ref))
