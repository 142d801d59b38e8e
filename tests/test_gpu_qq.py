"""GPU parity of the structurally different amplitudes (PAPER.md:87 last sentence): q qbar -> t tbar
and q qbar -> t tbar g against the CPU oracle, and the LO-multiprocess handle that reweights a mixed event list by process id."""
import numpy as np
import pytest

import oracle as orc
from paper_2312_07440_b200 import binding as B, events as ev

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
TOL64 = 1e-11


def rel(got, ref):
    return np.abs(got / ref - 1)


def gpu(process, po, pn, m, w, process_id=None, precision="fp64"):
    r = B.Reweighter(process, po, pn, precision)
    out = r.run(torch.from_numpy(np.ascontiguousarray(m)).cuda(), torch.from_numpy(np.ascontiguousarray(w)).cuda(), process_id=process_id)
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    r.close()
    return res


@pytest.mark.parametrize("idx,n", [(7, 4099), (8, 1203)])
def test_qqx_fp64_parity_every_event(idx, n):
    c = ev.config(idx)
    m, w = ev.generate(c, n)
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, m, w)
    got = gpu(c.process, c.params_old, c.params_new, m, w)
    for g, ref, name in zip(got, (a, b, wn), ("me_old", "me_new", "w_new")):
        e = rel(g, ref)
        assert e.max() < TOL64, (c.process, name, int(e.argmax()), e.max())
    same = gpu(c.process, c.params_new, c.params_new, m, w)
    assert np.array_equal(same[0], same[1]) and np.array_equal(same[2], w)


@pytest.mark.parametrize("idx,n", [(7, 1001), (8, 301)])
def test_qqx_several_sets_masses_and_rotated_frames(idx, n):
    c = ev.config(idx)
    m, w = ev.generate(c, n)
    rng = np.random.default_rng(idx)
    q, r = np.linalg.qr(rng.normal(size=(3, 3)))
    q = q @ np.diag(np.sign(np.diag(r)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    mr = m.copy()
    mr[:, 1:, :] = np.einsum("ab,pbn->pan", q, m[:, 1:, :])            # incoming legs off the axis
    for sets in ([c.params_new, ev.params(alpha_s=0.13, ggg_scale=0.8), c.params_old.copy()],
                 [ev.params(mt=170.0, ggg_scale=1.2), c.params_new, ev.params(mt=176.0)]):
        got = gpu(c.process, c.params_old, sets, mr, w)
        K = len(sets)
        for k, pn in enumerate(sets):
            a, b, wn, _ = orc.reweight(c.process, c.params_old, pn, mr, w)
            assert rel(got[0], a).max() < TOL64 and rel(got[1 + k], b).max() < TOL64 and rel(got[1 + K + k], wn).max() < TOL64


@pytest.mark.parametrize("procs,idxs,n,precision", [("gg_ttx,qqx_ttx", (2, 7), 3001, "fp64"), ("gg_ttxg,qqx_ttxg", (3, 8), 1501, "fp64"),
                                                   ("qqx_ttxg,gg_ttxg", (8, 3), 777, "fp32")])
def test_multiprocess_mixed_event_list(procs, idxs, n, precision):
    """One event list, two amplitudes (PAPER.md:127-131 'LO multiprocesses'): every event against the oracle of ITS process; the result
    equals what the single-process handles give on the sub-lists, bitwise."""
    rng = np.random.default_rng(n)
    pid = rng.integers(0, 2, size=n).astype(np.int32)
    cs = [ev.config(i) for i in idxs]
    parts = [ev.generate(c, n) for c in cs]
    m = np.where(pid[None, None, :] == 0, parts[0][0], parts[1][0])
    w = np.where(pid == 0, parts[0][1], parts[1][1])
    po, sets = ev.params(), [ev.params(ggg_scale=1.1, gggg_scale=1.1), ev.params(alpha_s=0.125, ggg_scale=0.9)]
    got = gpu(procs, po, sets, m, w, process_id=pid, precision=precision)
    K = len(sets)
    tol = TOL64 if precision == "fp64" else 1e-4
    for j, c in enumerate(cs):
        sel = np.nonzero(pid == j)[0]
        ms, ws = np.ascontiguousarray(m[:, :, sel]), w[sel].copy()
        for k, pn in enumerate(sets):
            a, b, wn, _ = orc.reweight(c.process, po, pn, ms, ws)
            assert rel(got[0, sel], a).max() < tol and rel(got[1 + k, sel], b).max() < tol and rel(got[1 + K + k, sel], wn).max() < tol
        single = gpu(c.process, po, sets, ms, ws, precision=precision if c.process.startswith("gg_ttxg") else "fp64")
        assert np.array_equal(single, got[:, sel])


def test_multiprocess_argument_errors():
    po, pn = ev.params(), [ev.params(ggg_scale=1.1)]
    with pytest.raises(RuntimeError, match="another number of external legs"):
        B.rwgt_create_multiprocess("gg_ttx,qqx_ttxg", po, pn)
    with pytest.raises(RuntimeError, match="QCD processes only"):
        B.rwgt_create_multiprocess("gg_ttx,epem_mupmum", po, pn)
    with pytest.raises(RuntimeError, match="unknown process"):
        B.rwgt_create_multiprocess("gg_ttx,nonsense", po, pn)
    h = B.rwgt_create_multiprocess("gg_ttx, qqx_ttx", po, pn)
    assert B.rwgt_n_processes(h) == 2 and B.rwgt_n_external(h) == 4 and B.rwgt_n_sets(h) == 1
    c = ev.config(2)
    m, w = ev.generate(c, 10)
    dm, dw, out = torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda(), torch.empty((3, 10), dtype=torch.float64, device="cuda")
    with pytest.raises(RuntimeError, match="process_id outside"):
        B.rwgt_run_multiprocess(h, dm.data_ptr(), dw.data_ptr(), np.full(10, 2, dtype=np.int32), out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), 10)
    with pytest.raises(RuntimeError, match="rwgt_run_multiprocess"):
        B.rwgt_run_multi(h, dm.data_ptr(), dw.data_ptr(), out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), 10)
    # all events of one process, none of the other
    B.rwgt_run_multiprocess(h, dm.data_ptr(), dw.data_ptr(), np.zeros(10, dtype=np.int32), out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), 10)
    torch.cuda.synchronize()
    a, b, wn, _ = orc.reweight("gg_ttx", po, pn[0], m, w)
    assert rel(out.cpu().numpy(), np.stack([a, b, wn])).max() < TOL64
    B.rwgt_destroy(h)
    h1 = B.rwgt_create("gg_ttx", po, pn[0])
    assert B.rwgt_n_processes(h1) == 1
    with pytest.raises(RuntimeError, match="not a multiprocess handle"):
        B.rwgt_run_multiprocess(h1, dm.data_ptr(), dw.data_ptr(), np.zeros(10, dtype=np.int32), out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), 10)
    B.rwgt_destroy(h1)
