"""CPU tests of the host-side logic: inputs, C-ABI exports, sharding (gloo, world_size 2), bench helpers."""
import ctypes
import json
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2312_07440_b200 import binding, events as ev, sharding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_events_deterministic_on_shell_and_conserving():
    for c in ev.CONFIGS:
        m1, w1 = ev.generate(c, 300)
        m2, w2 = ev.generate(c, 300)
        assert np.array_equal(m1, m2) and np.array_equal(w1, w2)
        assert m1.shape == (c.n_ext, 4, 300) and m1.flags.c_contiguous
        tot = m1[2:].sum(axis=0)
        assert np.abs(tot[0] - c.sqrts).max() < 1e-11 * c.sqrts and np.abs(tot[1:]).max() < 1e-11 * c.sqrts
        for k, mass in enumerate(c.final_masses):
            p = m1[2 + k]
            assert np.abs(p[0] ** 2 - (p[1:] ** 2).sum(0) - mass * mass).max() < 1e-9 * c.sqrts ** 2
        assert np.all(m1[0, 3] == c.sqrts / 2) and np.all(m1[1, 3] == -c.sqrts / 2) and np.all(m1[:2, 1:3] == 0)
        assert np.all(w1 > 0)
        # a prefix of a longer set is the shorter set (candidate stream, not block size, defines the events)
        m3, w3 = ev.generate(c, 50)
        assert np.array_equal(m3, m1[:, :, :50]) and np.array_equal(w3, w1[:50])


def test_event_cuts():
    for idx in (3, 4, 5):
        c = ev.config(idx)
        m, _ = ev.generate(c, 2000)
        g = m[4:]
        assert np.hypot(g[:, 1], g[:, 2]).min() > 20.0
        if c.dr_cut:
            y = 0.5 * np.log((g[:, 0] + g[:, 3]) / (g[:, 0] - g[:, 3]))
            ph = np.arctan2(g[:, 2], g[:, 1])
            for i in range(len(g)):
                for j in range(i + 1, len(g)):
                    d = np.abs(ph[i] - ph[j])
                    d = np.where(d > np.pi, 2 * np.pi - d, d)
                    assert np.hypot(y[i] - y[j], d).min() > 0.4


def test_weights_lognormal():
    _, w = ev.generate(ev.config(2), 200000)
    z = np.log(w)
    assert abs(z.mean()) < 0.01 and abs(z.std() - 1) < 0.01


def test_library_exports_every_declared_symbol():
    """Every include/*.h against the library that implements it and the binding that wraps it."""
    from paper_2312_07440_b200 import microbench
    headers = {"rwgt.h": (binding.LIB_PATH, binding.EXPORTS), "rwgt_microbench.h": (microbench.LIB_PATH, microbench.EXPORTS)}
    assert set(os.listdir(os.path.join(ROOT, "include"))) == set(headers)
    for hname, (libpath, exports) in headers.items():
        so = ctypes.CDLL(libpath)
        header = open(os.path.join(ROOT, "include", hname)).read()
        declared = set(re.findall(r"\b(rwgt_[a-z_0-9]+)\s*\(", header)) - {"rwgt_handle", "rwgt_params"}
        assert declared == set(exports), (hname, declared ^ set(exports))
        for name in declared:
            assert hasattr(so, name), name
            assert hasattr(binding if hname == "rwgt.h" else microbench, name), name
    # the measurement aid is not part of the product library
    assert not hasattr(ctypes.CDLL(binding.LIB_PATH), "rwgt_microbench_peak")


def test_host_only_entry_points_without_gpu():
    # colour matrix is host code; create must fail loudly (no CPU fallback) when no device is present
    C = binding.rwgt_colour_matrix(3)
    assert abs(C[0, 0] - 64 / 9) < 1e-15 and np.allclose(C, C.T)
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(RuntimeError, match="no CUDA device"):
            binding.rwgt_create("gg_ttx", ev.params(), ev.params())


def test_shard_bounds_cover_exactly():
    for n in (0, 1, 7, 1048576, 65537):
        for world in (1, 2, 3, 8):
            b = [sharding.shard_bounds(n, r, world) for r in range(world)]
            assert b[0][0] == 0 and b[-1][1] == n
            assert all(b[i][1] == b[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_bounds(10, 2, 2)


_GLOO = r"""
import os, sys, numpy as np, torch, torch.distributed as dist
sys.path.insert(0, %r)
from paper_2312_07440_b200 import events as ev, sharding
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d", rank=int(sys.argv[1]), world_size=2)
rank, world = dist.get_rank(), dist.get_world_size()
c = ev.config(3)
m, w = ev.generate(c, 101)
lo, hi = sharding.shard_bounds(101, rank, world)
# stand-in for the per-rank kernel: any per-event function of the shard (no exchange step exists)
sizes = [sharding.shard_bounds(101, r, world)[1] - sharding.shard_bounds(101, r, world)[0] for r in range(world)]
local = torch.zeros(max(sizes), dtype=torch.float64)
local[: hi - lo] = torch.from_numpy(w[lo:hi] * m[2, 0, lo:hi])
parts = [torch.zeros(max(sizes), dtype=torch.float64) for r in range(world)]
dist.all_gather(parts, local)
full = torch.cat([p[:s] for p, s in zip(parts, sizes)]).numpy()
assert np.array_equal(full, w * m[2, 0])
t = bench.max_over_ranks(0.5 + rank)       # slowest rank defines the time
assert t == 1.5
val = sharding.aggregate_throughput([hi - lo for lo, hi in (sharding.shard_bounds(101, r, world) for r in range(world))], 3, t)
assert abs(val - 101 * 3 / 1.5) < 1e-12
dist.barrier(); dist.destroy_process_group()
print("ok", rank)
"""


def test_two_rank_gloo_sharding_and_timing_reduction(tmp_path):
    port = 29500 + os.getpid() % 2000
    script = tmp_path / "gloo_rank.py"
    script.write_text(_GLOO % (ROOT, port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=240) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
        assert "ok" in o


def test_bench_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--ref-events", "512"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "events/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["config"]["workload"].startswith("gg_ttx")


def test_event_and_result_file_layout_round_trip(tmp_path):
    """The binary SoA files that stand in for LHE files (include/rwgt.h): 64-byte headers, planes in rwgt_run's layout."""
    c = ev.config(4)
    m, w = ev.generate(c, 33)
    f = str(tmp_path / "e.rwgt")
    binding.write_event_file(f, c.process, m, w)
    assert os.path.getsize(f) == 64 + (c.n_ext * 4 + 1) * 33 * 8
    raw = open(f, "rb").read()
    assert raw[:8] == b"RWGTEVT1" and int.from_bytes(raw[8:12], "little") == 1 and int.from_bytes(raw[12:16], "little") == c.n_ext
    assert int.from_bytes(raw[16:24], "little") == 33 and raw[24:24 + len(c.process)] == c.process.encode()
    assert np.array_equal(np.frombuffer(raw[64:64 + 33 * 8], dtype="<f8"), m[0, 0])       # first plane: E of leg 0
    p, m2, w2 = binding.read_event_file(f)
    assert p == c.process and np.array_equal(m2, m) and np.array_equal(w2, w)
    assert binding.event_file_n_events(f) == 33 and binding.event_file_process(f) == c.process
    # a result file as librwgt.so lays it out
    K, n = 2, 5
    hd = np.zeros(1, dtype=binding._RES_HDR)
    hd["magic"], hd["version"], hd["n_sets"], hd["n_events"], hd["process"], hd["first_event"] = b"RWGTRES1", 1, K, n, b"gg_ttxgg", 7
    body = np.arange((1 + 2 * K) * n + 1 + K, dtype=np.float64)
    r = str(tmp_path / "r.rwgt")
    open(r, "wb").write(hd.tobytes() + body.tobytes())
    res = binding.read_result_file(r)
    assert res["first_event"] == 7 and res["me_new"].shape == (K, n) and res["w_new"][1, 4] == 24.0 and res["sum_w_old"] == 25.0 and list(res["sum_w_new"]) == [26.0, 27.0]


def test_reweight_file_cli_parses_parameter_sets():
    from paper_2312_07440_b200 import reweight_file
    p = reweight_file.parse_set("ggg_scale=1.1,mt=170")
    assert p[ev.PARAM_NAMES.index("ggg_scale")] == 1.1 and p[ev.PARAM_NAMES.index("mt")] == 170.0 and p[ev.PARAM_NAMES.index("alpha_s")] == 0.118
    with pytest.raises(SystemExit):
        reweight_file.parse_set("nonsense=1")


def test_stored_full_set_goldens_are_the_oracle_values():
    """tests/golden/full_cfg<N>.npz hold every event of every config and are what the GPU parity tests compare with.
    They are written by tests/golden/make_goldens.py from the CPU oracle alone; this re-evaluates events sampled from the whole range
    with the oracle (never the CUDA path) and requires the stored numbers back, so a file of any other origin would show."""
    import oracle as orc
    gold = os.path.join(os.path.dirname(__file__), "golden")
    rng = np.random.default_rng(2312_07440)
    for idx, nsample in ((1, 64), (2, 64), (3, 24), (4, 8), (5, 2), (6, 6)):
        c = ev.config(idx)
        g = np.load(os.path.join(gold, f"full_cfg{idx}.npz"))
        out = g["out"]
        assert out.shape == (3, c.n_events) and np.all(np.isfinite(out)) and np.all(out[:2] > 0)
        assert int(g["seed"]) == c.seed and np.array_equal(g["params_old"], c.params_old) and np.array_equal(g["params_new"], c.params_new)
        m, w = ev.generate(c)
        pick = np.sort(rng.choice(c.n_events, size=nsample, replace=False))
        a, b, wn, _ = orc.reweight(c.process, c.params_old, c.params_new, np.ascontiguousarray(m[:, :, pick]), w[pick].copy())
        for k, ref in enumerate((a, b, wn)):
            # 2e-15: the oracle re-run gives the stored value back to the last bits (bit-exact for cfgs 1, 2, 6; a few ulp from the
            # summation order over threads for cfgs 3-5), whereas the FP64 kernels sit 1e-14..3e-13 away from it (profiles/r2_parity.md)
            assert np.abs(out[k, pick] / ref - 1).max() < 2e-15, (idx, k)


def test_stored_k_set_goldens_are_the_oracle_values():
    """tests/golden/ksets_cfg<N>_<list>.npz (make_goldens.py --sets): the stored lists and event indices are the ones events.py
    names, and sampled entries re-evaluated with the oracle give the stored numbers back (2e-15, as for the full-set files)."""
    import oracle as orc
    gold = os.path.join(os.path.dirname(__file__), "golden")
    rng = np.random.default_rng(7440)
    for idx, names in ev.KSET_GOLDENS.items():
        c = ev.config(idx)
        m, w = ev.generate(c)
        sel = ev.kset_sample(c)
        assert sel[0] == 0 and sel[-1] == c.n_events - 1 and np.all(np.diff(sel) > 0)
        full = np.load(os.path.join(gold, f"full_cfg{idx}.npz"))["out"]
        for name in names:
            g = np.load(os.path.join(gold, f"ksets_cfg{idx}_{name}.npz"))
            sets = ev.kset_list(c, name)
            assert np.array_equal(g["idx"], sel) and np.array_equal(g["sets"], np.array(sets)) and int(g["seed"]) == c.seed
            assert g["me_new"].shape == (len(sets), len(sel)) and np.all(np.isfinite(g["me_new"])) and np.all(g["me_new"] > 0)
            assert np.abs(g["me_old"] / full[0, sel] - 1).max() < 2e-15
            pick = np.sort(rng.choice(len(sel), size={3: 6, 4: 2, 5: 1}[idx], replace=False))
            k = int(rng.integers(len(sets)))
            a, b, wn, _ = orc.reweight(c.process, c.params_old, sets[k], np.ascontiguousarray(m[:, :, sel[pick]]), w[sel[pick]].copy())
            assert np.abs(g["me_new"][k, pick] / b - 1).max() < 2e-15 and np.abs(g["w_new"][k, pick] / wn - 1).max() < 2e-15, (idx, name, k)
