"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the same
seeded inputs.  Tolerances (BASELINE.json north_star / SURVEY Q9): FP64 1e-11 relative per event for each of
|M|^2, |M'|^2, W'; FP32 and mixed 1e-4 max, 1e-6 median."""
import numpy as np
import pytest

import oracle as orc
from paper_2312_07440_b200 import binding as B, events as ev

pytestmark = pytest.mark.gpu
TOL64 = 1e-11

torch = pytest.importorskip("torch")


def gpu_run(process, po, pn, m, w, precision="fp64", stream=None):
    r = B.Reweighter(process, po, pn, precision)
    dm, dw = torch.from_numpy(np.ascontiguousarray(m)).cuda(), torch.from_numpy(np.ascontiguousarray(w)).cuda()
    if stream is None:
        out = r.run(dm, dw)
    else:
        stream.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(stream):
            out = r.run(dm, dw)
        stream.synchronize()
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    r.close()
    return res


def rel(got, ref):
    return np.abs(got / ref - 1)


# sizes: several CTAs/slot groups plus a ragged tail, small enough for the oracle to finish in seconds
SMALL = {1: 4099, 2: 5003, 3: 1001, 4: 203, 5: 37}


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_fp64_parity_every_event_small(idx):
    c = ev.config(idx)
    m, w = ev.generate(c, SMALL[idx])
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, m, w)
    got = gpu_run(c.process, c.params_old, c.params_new, m, w)
    for g, ref, name in zip(got, (a, b, wn), ("me_old", "me_new", "w_new")):
        e = rel(g, ref)
        assert e.max() < TOL64, (c.process, name, int(e.argmax()), e.max())


@pytest.mark.parametrize("idx", [3, 4, 5])
@pytest.mark.parametrize("precision", ["fp32", "mixed"])
def test_fp32_and_mixed_parity(idx, precision):
    c = ev.config(idx)
    m, w = ev.generate(c, SMALL[idx])
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, m, w)
    got = gpu_run(c.process, c.params_old, c.params_new, m, w, precision)
    for g, ref in zip(got, (a, b, wn)):
        e = rel(g, ref)
        assert e.max() < 1e-4 and np.median(e) < 1e-6, (c.process, precision, e.max(), np.median(e))


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_full_size_bench_launch_sampled_against_oracle(idx):
    """BASELINE.json's full sizes in the launch configuration bench.py times; sampled events one by one."""
    c = ev.config(idx)
    m, w = ev.generate(c)
    assert w.shape[0] == c.n_events
    got = gpu_run(c.process, c.params_old, c.params_new, m, w)
    assert np.all(np.isfinite(got)) and np.all(got > 0)
    nsamp = {1: 64, 2: 64, 3: 48, 4: 12, 5: 6}[idx]
    rng = np.random.default_rng(100 + idx)
    sel = np.unique(np.concatenate([[0, c.n_events - 1], rng.integers(0, c.n_events, nsamp)]))
    for k in sel:
        p = np.ascontiguousarray(m[:, :, k])
        a, b = orc.me2(c.process, c.params_old, p), orc.me2(c.process, c.params_new, p)
        assert abs(got[0, k] / a - 1) < TOL64 and abs(got[1, k] / b - 1) < TOL64
        assert abs(got[2, k] / (w[k] * (b / a)) - 1) < TOL64
    # eq. 3 holds for every event of the full set
    assert np.all(np.abs(got[2] * got[0] - w * got[1]) <= 5e-16 * np.abs(w * got[1]))   # four roundings of 2^-53


@pytest.mark.parametrize("proc_idx", [(1, "epem_mupmum"), (2, "gg_ttx"), (2, "gg_ttx@bg"), (3, "gg_ttxg"), (4, "gg_ttxgg"), (5, "gg_ttxggg")])
def test_identical_parameter_sets_give_ratio_exactly_one(proc_idx):
    idx, proc = proc_idx
    c = ev.config(idx)
    m, w = ev.generate(c, min(SMALL[idx], 300))
    got = gpu_run(proc, c.params_new, c.params_new, m, w)
    assert np.array_equal(got[0], got[1]) and np.array_equal(got[2], w)


def test_generic_engine_agrees_with_dedicated_gg_ttx_kernel_and_oracle():
    c = ev.config(2)
    m, w = ev.generate(c, 3001)
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, m, w)
    g1 = gpu_run("gg_ttx", c.params_old, c.params_new, m, w)
    g2 = gpu_run("gg_ttx@bg", c.params_old, c.params_new, m, w)
    assert rel(g1, np.stack([a, b, wn])).max() < TOL64 and rel(g2, np.stack([a, b, wn])).max() < TOL64


@pytest.mark.parametrize("idx", [2, 3])
def test_general_coupling_change_alpha_s_and_both_scales(idx):
    """A new set that moves alpha_s and the two scales independently (masses equal: externals stay shared)."""
    c = ev.config(idx)
    m, w = ev.generate(c, 257)
    pn = ev.params(mt=173.0, ggg_scale=1.05, gggg_scale=0.9, alpha_s=0.125)
    po = ev.params(mt=173.0)
    a, b, wn, _ = orc.reweight(c.process, po, pn, m, w)
    got = gpu_run(c.process, po, pn, m, w)
    assert rel(got, np.stack([a, b, wn])).max() < TOL64


@pytest.mark.parametrize("proc_idx_n", [("gg_ttx", 2, 1031), ("gg_ttx@bg", 2, 517), ("gg_ttxg", 3, 301), ("gg_ttxgg", 4, 67), ("gg_ttxggg", 5, 9)])
@pytest.mark.parametrize("mt_new", [170.0, 176.5])
def test_top_mass_change_single_new_set(proc_idx_n, mt_new):
    """SURVEY 8(f) #4 (PAPER.md:87 last sentence: parameters inside the amplitudes): the new set has another top mass.  The events
    stay on the OLD mass shell (same phase space); spinors and propagators of the new set use m_t' with E from the
    input (reading Q8 / DESIGN.md R8), in the oracle and in the kernels alike.  One new set: gg_ttx takes gg_ttx_kernel's two_pass
    branch, the engine its separate-externals path."""
    proc, idx, n = proc_idx_n
    c = ev.config(idx)
    m, w = ev.generate(c, n)
    pn = ev.params(mt=mt_new, ggg_scale=1.1, gggg_scale=1.1)
    a, b, wn, _ = orc.reweight(c.process, c.params_old, pn, m, w)
    got = gpu_run(proc, c.params_old, pn, m, w)
    assert rel(got, np.stack([a, b, wn])).max() < TOL64
    assert np.abs(b / a - 1).max() > 1e-3                  # the mass change is macroscopic


def _rotation(seed):
    rng = np.random.default_rng(seed)
    q, r = np.linalg.qr(rng.normal(size=(3, 3)))
    q = q @ np.diag(np.sign(np.diag(r)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def _boost(m, beta):
    """Boost every momentum of m[n_ext,4,n] by the velocity vector beta."""
    b2 = float(beta @ beta)
    g = 1.0 / np.sqrt(1.0 - b2)
    bp = np.einsum("k,pkn->pn", beta, m[:, 1:, :])
    out = np.empty_like(m)
    out[:, 0, :] = g * (m[:, 0, :] + bp)
    out[:, 1:, :] = m[:, 1:, :] + ((g - 1.0) * bp / b2 + g * m[:, 0, :])[:, None, :] * beta[None, :, None]
    return out


@pytest.mark.parametrize("idx,n", [(1, 2003), (2, 2003), (3, 401), (4, 61), (6, 61)])
def test_rotated_events_against_oracle_incoming_legs_off_axis(idx, n):
    """The seeded sets have legs 0, 1 exactly on the z axis, so only the exact-axis branches of polvec / make_chi ever see the
    incoming legs.  A random SO(3) rotation of every event puts them on the generic branch (the library must
    not assume beams along z); compared with the oracle on the SAME rotated momenta, both parameter sets, and with the
    unrotated result (rotations are a symmetry of both sets, reading Q1)."""
    c = ev.config(idx)
    m, w = ev.generate(c, n)
    R = _rotation(40 + idx)
    mr = m.copy()
    mr[:, 1:, :] = np.einsum("ab,pbn->pan", R, m[:, 1:, :])
    assert np.abs(mr[0, 1:3, :]).min() > 1.0               # leg 0 has left the axis
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, mr, w)
    got = gpu_run(c.process, c.params_old, c.params_new, mr, w)
    assert rel(got, np.stack([a, b, wn])).max() < TOL64
    g0 = gpu_run(c.process, c.params_old, c.params_new, m, w)
    assert rel(got, g0).max() < 1e-10


@pytest.mark.parametrize("idx,n", [(1, 2003), (2, 2003), (3, 401), (4, 61), (6, 61)])
def test_boosted_events_against_oracle(idx, n):
    """A boost along a generic direction: legs 0, 1 off the axis and no longer back to back.  The oracle is evaluated on the same
    boosted momenta (for cfgs 2-4 the NEW set is frame dependent, reading Q1, so it is compared in the boosted frame only); the old
    set (and both sets of cfgs 1, 6) must also agree with the unboosted launch."""
    c = ev.config(idx)
    m, w = ev.generate(c, n)
    mb = _boost(m, np.array([0.21, -0.13, 0.32]))
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, mb, w)
    got = gpu_run(c.process, c.params_old, c.params_new, mb, w)
    assert rel(got, np.stack([a, b, wn])).max() < TOL64
    g0 = gpu_run(c.process, c.params_old, c.params_new, m, w)
    assert rel(got[0], g0[0]).max() < 1e-10
    if idx in (1, 6):
        assert rel(got[1], g0[1]).max() < 1e-10


def test_edge_cases_empty_single_and_bad_arguments():
    c = ev.config(3)
    h = B.rwgt_create(c.process, c.params_old, c.params_new)
    assert B.rwgt_n_external(h) == 5 and B.rwgt_flops_per_event(h) > 0
    B.rwgt_run(h, 0, 0, 0, 0, 0, 0)                      # n_events == 0: no-op, pointers not touched
    with pytest.raises(RuntimeError):
        B.rwgt_run(h, 0, 0, 0, 0, 0, 5)                  # NULL buffers
    with pytest.raises(RuntimeError):
        B.rwgt_run(h, 1, 1, 1, 1, 1, -1)
    B.rwgt_destroy(h)
    with pytest.raises(RuntimeError, match="unknown process"):
        B.rwgt_create("pp_jj", c.params_old, c.params_new)
    with pytest.raises(RuntimeError, match="invalid parameter"):
        B.rwgt_create(c.process, ev.params(alpha_s=-1.0), c.params_new)
    with pytest.raises(RuntimeError, match="invalid parameter"):
        B.rwgt_create(c.process, ev.params(Gamma_t=1.4), c.params_new)
    h1 = B.rwgt_create("epem_mupmum", ev.config(1).params_old, ev.config(1).params_new)
    with pytest.raises(RuntimeError, match="FP64 only"):
        B.rwgt_set_precision(h1, "fp32")
    B.rwgt_destroy(h1)
    for idx in (1, 2, 3, 5):
        cc = ev.config(idx)
        m, w = ev.generate(cc, 1)
        a, b, wn, _ = orc.reweight(cc.process, cc.params_old, cc.params_new, m, w)
        got = gpu_run(cc.process, cc.params_old, cc.params_new, m, w)
        assert rel(got[:, 0], np.array([a[0], b[0], wn[0]])).max() < TOL64


def test_zero_matrix_element_gives_ieee_result_no_error():
    """eq. 3 needs |M|^2 != 0.  Convention of include/rwgt.h: inf/nan is written, no error."""
    c = ev.config(2)
    m, w = ev.generate(c, 64)
    got = gpu_run(c.process, ev.params(alpha_s=1e-200), c.params_new, m, w)
    assert np.all(got[0] == 0) and np.all(~np.isfinite(got[2]))


def test_host_buffer_entry_point_and_non_default_stream():
    c = ev.config(3)
    m, w = ev.generate(c, 777)
    dev = gpu_run(c.process, c.params_old, c.params_new, m, w, stream=torch.cuda.Stream())
    h = B.rwgt_create(c.process, c.params_old, c.params_new)
    out = np.empty((3, 777))
    B.rwgt_run_host(h, m, w, out[0], out[1], out[2])
    B.rwgt_run_host(h, m[:, :, :100].copy(), w[:100].copy(), out[0, :100], out[1, :100], out[2, :100])
    B.rwgt_destroy(h)
    assert np.array_equal(out[:, 100:], dev[:, 100:]) and np.array_equal(out[:, :100], dev[:, :100])


def test_host_path_is_chunked_and_matches_device_path_bitwise():
    """rwgt_run_host cuts the events into overlapping copy/compute chunks (ragged last chunk, strided SoA planes):
    results must be bit-identical to one device launch, for pinned and pageable buffers."""
    for idx, n in ((1, 3 * 65536 + 123), (2, 2 * 65536 + 1), (3, 65536 + 77)):
        c = ev.config(idx)
        m0, w0 = ev.generate(c, 4096)
        reps = (n + 4095) // 4096
        m, w = np.tile(m0, (1, 1, reps))[:, :, :n].copy(), np.tile(w0, reps)[:n].copy()
        dev = gpu_run(c.process, c.params_old, c.params_new, m, w)
        h = B.rwgt_create(c.process, c.params_old, c.params_new)
        out = np.empty((3, n))
        B.rwgt_run_host(h, m, w, out[0], out[1], out[2])                       # pageable
        assert np.array_equal(out, dev)
        pm, pw, po = torch.from_numpy(m).pin_memory(), torch.from_numpy(w).pin_memory(), torch.empty((3, n), dtype=torch.float64).pin_memory()
        o = po.numpy()
        B.rwgt_run_host(h, pm.numpy(), pw.numpy(), o[0], o[1], o[2], torch.cuda.Stream().cuda_stream)
        assert np.array_equal(o, dev)
        B.rwgt_destroy(h)


def test_rotation_invariance_of_both_sets_on_gpu():
    """Property that holds at any size: a common spatial rotation leaves |M|^2 and |M'|^2 unchanged.
    Rotate about the beam axis so legs 0,1 stay on the exact-axis branch."""
    c = ev.config(4)
    m, w = ev.generate(c, 500)
    th = 0.7
    R = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    mr = m.copy()
    mr[:, 1:3, :] = np.einsum("ab,pbn->pan", R, m[:, 1:3, :])
    g0 = gpu_run(c.process, c.params_old, c.params_new, m, w)
    g1 = gpu_run(c.process, c.params_old, c.params_new, mr, w)
    assert rel(g1, g0).max() < 1e-10


@pytest.mark.parametrize("idx,n,precision", [(3, 4001, "fp64"), (3, 4001, "fp32"), (4, 1501, "fp64"), (4, 1501, "mixed"), (5, 301, "fp64"), (5, 301, "fp32"), (6, 3001, "fp64")])
def test_repeated_launches_are_bitwise_identical(idx, n, precision):
    """compute-sanitizer (racecheck) is not available on this pool: a race in the named-barrier hand-overs (worker / colour warps,
    staging buffers) or in the shared-memory tables would show up as run-to-run differences.  Same handle, same buffers, 6 launches,
    plus a fresh handle: all outputs bit-identical."""
    c = ev.config(idx)
    m, w = ev.generate(c, n)
    dm, dw = torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda()
    r = B.Reweighter(c.process, c.params_old, c.params_new, precision)
    ref = r.run(dm, dw).clone()
    for _ in range(5):
        out = r.run(dm, dw)
        torch.cuda.synchronize()
        assert torch.equal(out, ref)
    r.close()
    r2 = B.Reweighter(c.process, c.params_old, c.params_new, precision)
    assert torch.equal(r2.run(dm, dw), ref)
    r2.close()


def test_rwgt_run_can_be_captured_in_a_cuda_graph():
    """rwgt_run only enqueues one kernel on the caller's stream (no allocation, no sync, no copy: SURVEY 8(b)), so a launch-bound loop
    over small event sets can be captured once and replayed."""
    for idx, n in ((1, 16384), (3, 1001), (6, 257)):
        c = ev.config(idx)
        m, w = ev.generate(c, n)
        dm, dw = torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda()
        r = B.Reweighter(c.process, c.params_old, c.params_new, "fp64")
        ref = r.run(dm, dw).clone()
        out = torch.zeros_like(ref)
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            r.run(dm, dw, out)                      # warm-up on the capture stream
        torch.cuda.current_stream().wait_stream(side)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            r.run(dm, dw, out)
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, ref)
        dw.mul_(2.0)                                # new inputs in the same buffers
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out[2], 2.0 * ref[2]) and torch.equal(out[0], ref[0])
        r.close()
