"""GPU test of rwgt_sum_weights_static, the one entry point of librwgt.so that allocates nothing (include/rwgt.h).

It is there for programs that cannot let a library call cudaMalloc: a generator or analysis framework that has taken all device
memory into its own arena (an allocation from a plug-in fails, or escapes the arena's accounting), and loops that cannot afford the
device-wide wait a cudaMalloc / cudaFree brings.  The eq. 2 sums are the same kernel as rwgt_sum_weights, with the
block partials and row counters in a fixed 9 KB array of the library image instead of a handle's buffers.

What is checked: the sums of the static entry point equal those of the handle path (which the other tests pin against exactly
rounded sums and the oracle) bitwise, and sit inside the error bound test_gpu_files.py uses, on two calls in a row that share the
static array: the second call has other data, another length and fewer rows, so anything the first call left behind would show.
The file is named to be collected last: pytest -x stops at the first failure and must not hide the parity tests behind this one.
It passes alone in a fresh process (the first call then does the per-device address lookup) and after the other tests.
"""
import math

import numpy as np
import pytest

from paper_2312_07440_b200 import binding as B, events as ev

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def handle_sums(rows_dev):
    """the existing path: a handle's rwgt_sum_weights (scratch allocated by rwgt_create)"""
    c = ev.config(1)
    r = B.Reweighter(c.process, c.params_old, c.params_new)
    s = r.cross_sections(rows_dev).cpu().numpy()
    r.close()
    return s


def static_sums(rows_dev):
    out = torch.full((rows_dev.shape[0],), float("nan"), dtype=torch.float64, device=rows_dev.device)
    B.rwgt_sum_weights_static(rows_dev.data_ptr(), rows_dev.shape[0], rows_dev.shape[1], out.data_ptr(),
                              torch.cuda.current_stream(rows_dev.device).cuda_stream)
    return out.cpu().numpy()


def test_static_sums_equal_the_handle_path_on_two_calls_in_a_row():
    rng = np.random.default_rng(20231207)
    calls = []
    for n_rows, n in ((B.RWGT_STATIC_SUM_MAX_ROWS, 300007), (3, 70001)):     # ragged lengths, the maximum number of rows first
        rows = np.exp(rng.normal(size=(n_rows, n)))
        rows[-1] *= np.where(rng.random(n) < 0.3, -1.0, 1.0)                   # some negative weights
        calls.append(rows)
    dev = [torch.from_numpy(r).cuda() for r in calls]
    got = [static_sums(d) for d in dev]                                        # two calls in a row on one stream, nothing between
    for rows, d, s in zip(calls, dev, got):
        want = handle_sums(d)
        assert np.array_equal(s, want)                                         # same partition, same trees: bitwise
        n = rows.shape[1]
        for k in range(rows.shape[0]):                                         # and the bound of test_gpu_files.py against the exact sum
            bound = (n / 16384 + 30) * 2.0 ** -53 * math.fsum(np.abs(rows[k]))
            assert abs(s[k] - math.fsum(rows[k])) <= bound
    # a third call repeats the first: the array's leftovers from call two change nothing
    assert np.array_equal(static_sums(dev[0]), got[0])


def test_static_sums_of_an_empty_row_and_of_one_event():
    d = torch.tensor([[1.5], [-2.25]], dtype=torch.float64, device="cuda")
    assert np.array_equal(static_sums(d), np.array([1.5, -2.25]))
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    B.rwgt_sum_weights_static(d.data_ptr(), 2, 0, out.data_ptr(), torch.cuda.current_stream().cuda_stream)   # n_events = 0: sums are 0
    assert np.array_equal(out.cpu().numpy(), np.zeros(2))


def test_static_sums_refuse_what_the_fixed_array_cannot_hold():
    d = torch.ones((1, 8), dtype=torch.float64, device="cuda")
    o = torch.zeros(32, dtype=torch.float64, device="cuda")
    with pytest.raises(RuntimeError, match="n_rows outside 1..RWGT_STATIC_SUM_MAX_ROWS"):
        B.rwgt_sum_weights_static(d.data_ptr(), B.RWGT_STATIC_SUM_MAX_ROWS + 1, 8, o.data_ptr())
    with pytest.raises(RuntimeError, match="n_rows"):
        B.rwgt_sum_weights_static(d.data_ptr(), 0, 8, o.data_ptr())
    with pytest.raises(RuntimeError, match="NULL"):
        B.rwgt_sum_weights_static(0, 1, 8, o.data_ptr())
    with pytest.raises(RuntimeError, match="n_events"):
        B.rwgt_sum_weights_static(d.data_ptr(), 1, -1, o.data_ptr())
    # a refused call leaves the entry point usable
    assert static_sums(d)[0] == 8.0
