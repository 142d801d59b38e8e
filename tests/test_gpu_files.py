"""GPU tests of the host side of the procedure (PAPER.md:87 steps 2 and 8): binary SoA event files through
rwgt_run_file, and the eq. 2 sums of rwgt_sum_weights."""
import math
import os

import numpy as np
import pytest

import oracle as orc
from paper_2312_07440_b200 import binding as B, events as ev

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def device_run(c, sets, m, w):
    r = B.Reweighter(c.process, c.params_old, sets)
    out = r.run(torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda()).cpu().numpy()
    r.close()
    return out


@pytest.mark.parametrize("idx,n,K", [(1, 70001, 2), (2, 200003, 1), (3, 40961, 3), (6, 5000, 2)])
def test_run_file_matches_device_path_bitwise_and_oracle_sums(tmp_path, idx, n, K):
    c = ev.config(idx)
    m0, w0 = ev.generate(c, min(n, 8192))
    reps = (n + m0.shape[2] - 1) // m0.shape[2]
    m, w = np.tile(m0, (1, 1, reps))[:, :, :n].copy(), np.tile(w0, reps)[:n].copy()
    sets = [c.params_new, c.params_old.copy(), ev.params(alpha_em=1 / 120.0, alpha_s=0.125, ggg_scale=0.9)][:K]
    fin, fout = str(tmp_path / "events.rwgt"), str(tmp_path / "results.rwgt")
    B.write_event_file(fin, c.process, m, w)
    h = B.rwgt_create_multi(c.process, c.params_old, sets)
    B.rwgt_run_file(h, fin, fout)
    res = B.read_result_file(fout)
    dev = device_run(c, sets, m, w)
    assert res["process"] == c.process and res["first_event"] == 0
    assert np.array_equal(res["me_old"], dev[0]) and np.array_equal(res["me_new"], dev[1:1 + K]) and np.array_equal(res["w_new"], dev[1 + K:])
    # eq. 2 of the old weights and of every set, against exactly rounded sums of the file's own rows
    assert abs(res["sum_w_old"] / math.fsum(w) - 1) < 1e-13
    for k in range(K):
        assert abs(res["sum_w_new"][k] / math.fsum(res["w_new"][k]) - 1) < 1e-13
    if K >= 2:
        assert res["sum_w_new"][1] == res["sum_w_old"]            # the set equal to the old one: same weights, same summation tree
    # a sub-range, as a rank of a multi-GPU job would take it; second call reuses the handle's buffers
    lo, cnt = n // 3, n // 2
    B.rwgt_run_file(h, fin, fout, lo, cnt)
    part = B.read_result_file(fout)
    assert part["first_event"] == lo and np.array_equal(part["w_new"], dev[1 + K:, lo:lo + cnt]) and np.array_equal(part["me_old"], dev[0, lo:lo + cnt])
    B.rwgt_destroy(h)


def test_run_file_against_the_oracle_every_event(tmp_path):
    c = ev.config(3)
    m, w = ev.generate(c, 1201)
    fin, fout = str(tmp_path / "e.rwgt"), str(tmp_path / "r.rwgt")
    B.write_event_file(fin, c.process, m, w)
    h = B.rwgt_create(c.process, c.params_old, c.params_new)
    B.rwgt_run_file(h, fin, fout)
    B.rwgt_destroy(h)
    res = B.read_result_file(fout)
    a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, m, w)
    assert np.abs(res["me_old"] / a - 1).max() < 1e-11 and np.abs(res["me_new"][0] / b - 1).max() < 1e-11 and np.abs(res["w_new"][0] / wn - 1).max() < 1e-11
    assert abs(res["sum_w_new"][0] / orc.cross_section(wn) - 1) < 1e-11 and abs(res["sum_w_old"] / orc.cross_section(w) - 1) < 1e-12


def test_run_file_error_behaviour(tmp_path):
    c = ev.config(2)
    m, w = ev.generate(c, 100)
    fin = str(tmp_path / "e.rwgt")
    B.write_event_file(fin, c.process, m, w)
    h3 = B.rwgt_create("gg_ttxg", c.params_old, c.params_new)
    with pytest.raises(RuntimeError, match="another process"):
        B.rwgt_run_file(h3, fin, str(tmp_path / "o.rwgt"))
    B.rwgt_destroy(h3)
    h = B.rwgt_create(c.process, c.params_old, c.params_new)
    with pytest.raises(RuntimeError, match="cannot open"):
        B.rwgt_run_file(h, str(tmp_path / "missing.rwgt"), str(tmp_path / "o.rwgt"))
    with pytest.raises(RuntimeError, match="range outside"):
        B.rwgt_run_file(h, fin, str(tmp_path / "o.rwgt"), 50, 51)
    with open(fin, "r+b") as f:
        f.truncate(64 + 100 * 8 * 5)
    with pytest.raises(RuntimeError, match="truncated"):
        B.rwgt_run_file(h, fin, str(tmp_path / "o.rwgt"))
    bad = str(tmp_path / "bad.rwgt")
    open(bad, "wb").write(b"x" * 200)
    with pytest.raises(RuntimeError, match="not an event file"):
        B.rwgt_run_file(h, bad, str(tmp_path / "o.rwgt"))
    B.write_event_file(fin, c.process, m[:, :, :0].copy(), w[:0].copy())          # empty file: valid, empty result
    B.rwgt_run_file(h, fin, str(tmp_path / "o.rwgt"))
    res = B.read_result_file(str(tmp_path / "o.rwgt"))
    assert res["me_old"].shape == (0,) and res["sum_w_old"] == 0.0
    B.rwgt_destroy(h)


def test_run_file_never_destroys_the_input_and_leaves_no_result_after_a_failure(tmp_path):
    """out_path == in_path is refused with the event file intact; a header whose n_events would wrap the size product counts as
    truncated; a failed call leaves neither a result file nor its ".tmp", and an earlier result of the same name stays as it was."""
    c = ev.config(2)
    m, w = ev.generate(c, 300)
    fin, fout = str(tmp_path / "e.rwgt"), str(tmp_path / "o.rwgt")
    B.write_event_file(fin, c.process, m, w)
    before = open(fin, "rb").read()
    h = B.rwgt_create(c.process, c.params_old, c.params_new)
    with pytest.raises(RuntimeError, match="event file itself"):
        B.rwgt_run_file(h, fin, fin)
    os.link(fin, str(tmp_path / "alias.rwgt"))                                 # the same inode under another name
    with pytest.raises(RuntimeError, match="event file itself"):
        B.rwgt_run_file(h, fin, str(tmp_path / "alias.rwgt"))
    assert open(fin, "rb").read() == before
    B.rwgt_run_file(h, fin, fout)                                              # a good result ...
    good = open(fout, "rb").read()
    assert not os.path.exists(fout + ".tmp")
    huge = str(tmp_path / "huge.rwgt")
    hd = bytearray(before[:64])
    hd[16:24] = (2 ** 61 + 5).to_bytes(8, "little")                            # (planes + 1) * n * 8 wraps to a small number
    open(huge, "wb").write(bytes(hd) + before[64:])
    with pytest.raises(RuntimeError, match="truncated"):
        B.rwgt_run_file(h, huge, fout)
    with pytest.raises(RuntimeError, match="range outside"):
        B.rwgt_run_file(h, fin, fout, 2 ** 62, 2 ** 62)                        # first + n wraps
    assert open(fout, "rb").read() == good and not os.path.exists(fout + ".tmp")   # ... survives the failed calls
    os.chmod(tmp_path, 0o500)                                                  # a directory that takes no new file
    try:
        if not os.access(str(tmp_path), os.W_OK):                              # (root ignores the mode: nothing to check then)
            with pytest.raises(RuntimeError, match="cannot create"):
                B.rwgt_run_file(h, fin, str(tmp_path / "new.rwgt"))
            assert not os.path.exists(str(tmp_path / "new.rwgt"))
    finally:
        os.chmod(tmp_path, 0o700)
    B.rwgt_destroy(h)


def test_set_precision_on_a_multiprocess_handle_without_fp32_members_is_refused():
    c = ev.config(2)
    h = B.rwgt_create_multiprocess("gg_ttx,qqx_ttx", c.params_old, [c.params_new])
    with pytest.raises(RuntimeError, match="FP64 only"):
        B.rwgt_set_precision(h, B.RWGT_FP32)
    B.rwgt_set_precision(h, B.RWGT_FP64)
    B.rwgt_destroy(h)
    h = B.rwgt_create_multiprocess("gg_ttxg,qqx_ttxg", c.params_old, [c.params_new])
    B.rwgt_set_precision(h, B.RWGT_MIXED)                                      # gg_ttxg has the mode; qqx_ttxg stays FP64
    B.rwgt_destroy(h)


@pytest.mark.parametrize("n", [1, 63, 64, 65, 16384, 1048576 + 17])
def test_sum_weights_deterministic_and_accurate(n):
    """eq. 2 on the device: within the documented bound of the exactly rounded sum, identical on repeated launches, equal to the
    oracle's plain sum to the same bound; rows are independent."""
    rng = np.random.default_rng(n)
    rows = np.exp(rng.normal(size=(3, n)))
    rows[2] *= np.where(rng.random(n) < 0.3, -1.0, 1.0)       # some negative weights
    c = ev.config(1)
    r = B.Reweighter(c.process, c.params_old, c.params_new)
    d = torch.from_numpy(rows).cuda()
    s1 = r.cross_sections(d).cpu().numpy()
    s2 = r.cross_sections(d).cpu().numpy()
    s3 = r.cross_sections(d[1:].contiguous()).cpu().numpy()
    r.close()
    assert np.array_equal(s1, s2) and np.array_equal(s1[1:], s3)
    for k in range(3):
        bound = (n / 16384 + 30) * 2.0 ** -53 * math.fsum(np.abs(rows[k]))
        assert abs(s1[k] - math.fsum(rows[k])) <= bound
        assert abs(s1[k] - orc.cross_section(rows[k])) <= bound + n * 2.0 ** -53 * math.fsum(np.abs(rows[k]))


def test_sum_weights_bad_arguments():
    c = ev.config(1)
    h = B.rwgt_create(c.process, c.params_old, c.params_new)
    with pytest.raises(RuntimeError, match="NULL"):
        B.rwgt_sum_weights(h, 0, 1, 5, 0)
    with pytest.raises(RuntimeError, match="n_rows"):
        B.rwgt_sum_weights(h, 8, B.RWGT_MAX_SETS + 2, 5, 8)
    B.rwgt_destroy(h)
