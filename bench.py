#!/usr/bin/env python
"""bench.py — reweighted events/s of the LO reweighting hot path (eq. 3; PAPER.md:87 steps 3-6).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--precision fp64] [--impl reference]
    python bench.py --sweep [--config 6]        # the paper's Fig. 2 / Fig. 3 axes, markdown tables
    python bench.py --parity-report             # max / median error against tests/golden/full_cfg*.npz, markdown table

A step = one pass of the whole hot path (one rwgt_run launch: a1-a7 of SURVEY §8(a)) over the synthetic
event set of one BASELINE.json config.  Default: configs[4] = gg -> ttbar ggg, 65,536 events, FP64: the largest
work per step and the config north_star's FMA-peak target is written on.  Every other config / precision is timed
with the same --steps / --warmup and reported inside the line (roofline.per_config, other_configs).  Prints ONE
JSON line (rank 0).  N > 1: launched by torchrun, every rank runs the same-size workload with its own seed
(weak scaling, no data-path collective: events are independent).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2312_07440_b200 import events as ev, sharding  # noqa: E402

# B200 plain-ALU peaks: 148 SMs x 4 SMSP x 16 FP64 (32 FP32) FMA lanes x 2 flop x clock
SM_COUNT = 148
FP64_LANES_PER_SM = 64
FP32_LANES_PER_SM = 128


def alu_peak_tflops(dtype: str, mhz: float) -> float:
    lanes = FP64_LANES_PER_SM if dtype == "f64" else FP32_LANES_PER_SM
    return SM_COUNT * lanes * 2 * mhz * 1e6 / 1e12


def measured_peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


def max_over_ranks(seconds: float) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return seconds
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([seconds], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
            time.sleep(0.15)
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.06)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self) -> dict:
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def workload_name(c: ev.Config, n: int) -> str:
    return f"{c.process} cfg{c.index} n={n} sqrt(s)={c.sqrts:g}"


def bytes_per_event(c: ev.Config) -> int:
    return (c.n_ext * 4 + 1) * 8 + 24          # SoA momenta + weight in, three doubles out


# ------------------------------------------------------------------------------------------------- reference arm
def run_reference(args) -> None:
    """The oracle, as it stands, timed on the host cores (tier rule: the reference arm IS the oracle)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as orc
    c = ev.config(args.config)
    cores = os.cpu_count() or 1
    n = args.ref_events or max(8, int(ORACLE_PER_CORE[c.index] * cores * 3.0))    # ~3 s per step
    n = min(n, c.n_events)
    m, w = ev.generate(c, n)
    for _ in range(args.warmup):
        orc.reweight(c.process, c.params_old, c.params_new, m, w)
    t0 = time.perf_counter()
    used = cores
    for _ in range(args.steps):
        _, _, _, used = orc.reweight(c.process, c.params_old, c.params_new, m, w)
    dt = (time.perf_counter() - t0) / args.steps
    val = n / dt
    sample = f"first {n} events of the seeded {workload_name(c, c.n_events)} set per step"
    line = {"impl": "reference", "metric": "reweighted events/s (both |M|^2)", "value": val, "unit": "events/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(c, c.n_events), "sample_events_per_step": n},
            "cpu_baseline": {"value": val, "unit": "events/s", "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------- our arm
def time_config(torch, B, c, precision, n, steps, warmup, seed_offset, flush_buf, sampler_index=None, tile_from=0, new_sets=None):
    """Device-resident timing of one config. Returns dict with per-step ms list etc."""
    if tile_from and tile_from < n:
        m0, w0 = ev.generate(c, tile_from, seed=c.seed + 1000 * seed_offset)
        reps = (n + tile_from - 1) // tile_from
        m, w = np.tile(m0, (1, 1, reps))[:, :, :n].copy(), np.tile(w0, reps)[:n].copy()
    else:
        m, w = ev.generate(c, n, seed=c.seed + 1000 * seed_offset)
    dm, dw = torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda()
    k_sets = len(new_sets) if new_sets else 1
    out = torch.empty((1 + 2 * k_sets, n), dtype=torch.float64, device="cuda")
    r = B.Reweighter(c.process, c.params_old, new_sets if new_sets else c.params_new, precision)
    stream = torch.cuda.current_stream()
    in_bytes = dm.numel() * 8 + dw.numel() * 8 + out.numel() * 8
    need_flush = in_bytes < 2 * 126e6
    for _ in range(warmup):
        r.run(dm, dw, out)
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for s0, s1 in evs:
        if need_flush:
            flush_buf.add_(1.0)                       # 512 MB read+write: evicts L2 between timed iterations
        s0.record(stream)
        r.run(dm, dw, out)
        s1.record(stream)
    torch.cuda.synchronize()
    ms = [a.elapsed_time(b) for a, b in evs]
    res = {"ms": ms, "flops_per_event": r.flops_per_event(), "tensor_flops_per_event": r.tensor_flops_per_event(), "out": out, "dm": dm, "dw": dw, "host": (m, w), "rw": r,
           "l2": "flushed between iterations (512 MB add_)" if need_flush else "inputs+outputs exceed L2 (no flush)"}
    return res


def per_config_entry(cc, prec, rr, max_mhz, hbm_peak):
    kms = statistics.mean(rr["ms"])
    dt_ = "f64" if prec == "fp64" else "f32"
    fpe = rr["flops_per_event"] + (rr["tensor_flops_per_event"] if dt_ == "f64" else 0.0)
    n = rr["n"]
    tf = fpe * n / (kms * 1e-3) / 1e12
    gbs = bytes_per_event(cc) * n / (kms * 1e-3) / 1e9
    return {"cfg": cc.index, "process": cc.process, "precision": prec, "n": n, "kernel_ms": round(kms, 5), "events_per_s": n / (kms * 1e-3),
            "alu_tflops": round(tf, 3), "alu_frac": round(tf / alu_peak_tflops(dt_, max_mhz), 4), "hbm_gbs": round(gbs, 1), "hbm_frac": round(gbs / hbm_peak, 4)}


def run_sweep(args) -> None:
    """The paper's two experiments (Fig. 2: runtime against the number of events for one parameter set; PAPER.md:117
    Fig. 3: runtime against the number of parameter sets), every point the mean (min-max) of 5 runs as in the paper.
    device = rwgt_run_multi on device-resident buffers (CUDA events); host = rwgt_run_multi_host on pinned host buffers, copies inside the
    timed call (the transfer overhead the paper describes for small n); file = rwgt_run_file, read + copy + kernel + write."""
    import tempfile
    import torch
    from paper_2312_07440_b200 import binding as B
    c = ev.config(args.config if args.config else 6)
    nmax = max(1 << args.max_log2, args.fig3_events)
    m0, w0 = ev.generate(c, min(nmax, c.n_events))
    reps = (nmax + m0.shape[2] - 1) // m0.shape[2]
    m = np.tile(m0, (1, 1, reps))[:, :, :nmax].copy()
    w = np.tile(w0, reps)[:nmax].copy()
    rng = np.random.default_rng(c.seed)
    tmp = tempfile.mkdtemp(prefix="rwgt_sweep_")

    def new_sets(k):
        if c.index == 6:      # a random electroweak coupling per set
            return [ev.params(alpha_em=float(a)) for a in rng.uniform(0.5, 2.0, size=k) / 132.5]
        if c.index == 1:
            return [ev.params(GammaZ=float(g), sin2_thetaW=float(x)) for g, x in zip(rng.uniform(2.3, 2.7, size=k), rng.uniform(0.22, 0.24, size=k))]
        return [ev.params(ggg_scale=float(1 + x), gggg_scale=float(1 + x)) for x in rng.uniform(-0.2, 0.2, size=k)]

    def stats(ts):
        return f"{np.mean(ts):.4f} ({min(ts):.4f}-{max(ts):.4f})"

    def measure(n, K):
        sets = new_sets(K)
        h = B.rwgt_create_multi(c.process, c.params_old, sets)
        mh = torch.from_numpy(np.ascontiguousarray(m[:, :, :n])).pin_memory()
        wh = torch.from_numpy(w[:n].copy()).pin_memory()
        dm, dw = mh.cuda(), wh.cuda()
        a = torch.empty(n, dtype=torch.float64, device="cuda")
        b = torch.empty((K, n), dtype=torch.float64, device="cuda")
        o = torch.empty((K, n), dtype=torch.float64, device="cuda")
        ha, hb, ho = torch.empty(n, dtype=torch.float64).pin_memory(), torch.empty((K, n), dtype=torch.float64).pin_memory(), torch.empty((K, n), dtype=torch.float64).pin_memory()
        st = torch.cuda.current_stream().cuda_stream
        fin, fout = os.path.join(tmp, "in.rwgt"), os.path.join(tmp, "out.rwgt")
        B.write_event_file(fin, c.process, mh.numpy(), wh.numpy())
        dev, host, fil = [], [], []
        for it in range(2 + 5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            B.rwgt_run_multi(h, dm.data_ptr(), dw.data_ptr(), a.data_ptr(), b.data_ptr(), o.data_ptr(), n, st)
            e1.record()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            B.rwgt_run_multi_host(h, mh.numpy(), wh.numpy(), ha.numpy(), hb.numpy(), ho.numpy())
            t1 = time.perf_counter()
            B.rwgt_run_file(h, fin, fout)
            t2 = time.perf_counter()
            if it >= 2:
                dev.append(e0.elapsed_time(e1)); host.append((t1 - t0) * 1e3); fil.append((t2 - t1) * 1e3)
        assert np.array_equal(ho.numpy(), o.cpu().numpy())
        res = B.read_result_file(fout)
        assert np.array_equal(res["w_new"], ho.numpy())
        B.rwgt_destroy(h)
        return dev, host, fil

    print(f"# {c.process} (config {c.index}), FP64\n")
    print("## Runtime against the number of events, one parameter set (PAPER.md:105 Fig. 2), ms: mean (min-max) of 5\n")
    print("| events | device ms | host-buffer ms | file ms (read + copy + kernel + write) | device events/s | host-buffer events/s | file events/s |\n|---|---|---|---|---|---|---|")
    for lg in range(0, args.max_log2 + 1, 2):
        n = 1 << lg
        dev, host, fil = measure(n, 1)
        print(f"| {n} | {stats(dev)} | {stats(host)} | {stats(fil)} | {n / np.mean(dev) * 1e3:.3e} | {n / np.mean(host) * 1e3:.3e} | {n / np.mean(fil) * 1e3:.3e} |", flush=True)
    n = args.fig3_events
    print(f"\n## Runtime against the number of parameter sets, {n} events (PAPER.md:117 Fig. 3), ms: mean (min-max) of 5\n")
    print("| parameter sets | device ms | host-buffer ms | file ms | new weights/s (device) |\n|---|---|---|---|---|")
    for K in [int(x) for x in args.sets.split(",")]:
        dev, host, fil = measure(n, K)
        print(f"| {K} | {stats(dev)} | {stats(host)} | {stats(fil)} | {K * n / np.mean(dev) * 1e3:.3e} |", flush=True)


def run_parity_report(args) -> None:
    """Per config and precision: max / median relative error of |M|^2, |M'|^2, W' of the full-size launch against the stored oracle
    values tests/golden/full_cfg<N>.npz (written by tests/golden/make_goldens.py from the CPU oracle alone), events over tolerance,
    worst event.  Reads files only: the oracle is not executed."""
    import torch
    from paper_2312_07440_b200 import binding as B
    tol = {"fp64": (1e-11, 1e-11), "fp32": (1e-4, 1e-6), "mixed": (1e-4, 1e-6)}
    print("| cfg | process | precision | events compared (of the launch) | output | max rel. err | median rel. err | tolerance (max / median) | events over max tolerance | worst event |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for idx in (1, 2, 3, 4, 5, 6):
        c = ev.config(idx)
        f = os.path.join(ROOT, "tests", "golden", f"full_cfg{idx}.npz")
        if not os.path.exists(f):
            print(f"| {idx} | {c.process} | - | golden file missing | | | | | | |")
            continue
        ref = np.load(f)["out"]
        ng = ref.shape[1]
        m, w = ev.generate(c)
        dm, dw = torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda()
        for prec in c.precisions + (("mixed",) if "fp32" in c.precisions else ()):
            r = B.Reweighter(c.process, c.params_old, c.params_new, prec)
            got = r.run(dm, dw).cpu().numpy()
            r.close()
            tmax, tmed = tol[prec]
            for k, name in enumerate(("|M|^2", "|M'|^2", "W'")):
                e = np.abs(got[k, :ng] / ref[k] - 1)
                print(f"| {idx} | {c.process} | {prec} | {ng} ({c.n_events}) | {name} | {e.max():.2e} | {np.median(e):.2e} | {tmax:g} / {tmed:g} | {int((e > tmax).sum())} | {int(e.argmax())} |", flush=True)
    # K new parameter sets per pass (PAPER.md:87 step 7): full-size launches with the named lists of events.kset_list against the oracle values of
    # tests/golden/ksets_cfg<N>_<list>.npz on the multi-round sample events.kset_sample; one row per (cfg, list, precision, set)
    print()
    print("| cfg | list | K | precision | set | events compared (of the launch) | max rel. err |M'_k|^2 | median | max rel. err W'_k | median | tolerance (max / median) | over tolerance | old == new bitwise |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for idx, names in ev.KSET_GOLDENS.items():
        c = ev.config(idx)
        m, w = ev.generate(c)
        dm, dw = torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda()
        for lname in names:
            f = os.path.join(ROOT, "tests", "golden", f"ksets_cfg{idx}_{lname}.npz")
            if not os.path.exists(f):
                print(f"| {idx} | {lname} | - | - | - | golden file missing | | | | | | | |")
                continue
            g = np.load(f)
            sets, sel = ev.kset_list(c, lname), g["idx"]
            K = len(sets)
            for prec in ("fp64", "fp32", "mixed"):
                r = B.Reweighter(c.process, c.params_old, sets, prec)
                got = r.run(dm, dw).cpu().numpy()
                r.close()
                tmax, tmed = tol[prec]
                for k in range(K):
                    eb, ew = np.abs(got[1 + k, sel] / g["me_new"][k] - 1), np.abs(got[1 + K + k, sel] / g["w_new"][k] - 1)
                    same = "-"
                    if np.array_equal(sets[k], c.params_old):
                        same = "yes (all events)" if np.array_equal(got[1 + k], got[0]) and np.array_equal(got[1 + K + k], w) else "NO"
                    print(f"| {idx} | {lname} | {K} | {prec} | {k} | {len(sel)} ({c.n_events}) | {eb.max():.2e} | {np.median(eb):.2e} | {ew.max():.2e} | {np.median(ew):.2e} | "
                          f"{tmax:g} / {tmed:g} | {int((eb > tmax).sum() + (ew > tmax).sum())} | {same} |", flush=True)


# rough oracle events/s/core (both parameter sets), measured on this pool's hosts; only sizes the bounded CPU samples
ORACLE_PER_CORE = {1: 150000.0, 2: 6000.0, 3: 300.0, 4: 25.0, 5: 1.8, 6: 25.0, 7: 3000.0, 8: 150.0}


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=0, help="BASELINE.json config index 1..5 (default 5 = configs[4], the config north_star's FMA target names); "
                                                          "6 = the paper's own e+e- -> 5 gamma (PAPER.md:72-77)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "mixed"])
    ap.add_argument("--events", type=int, default=0, help="override the config's event count")
    ap.add_argument("--ref-events", type=int, default=0, help="reference arm: events per step")
    ap.add_argument("--no-extra", action="store_true", help="skip the other configs / precisions")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="throughput against events / parameter sets (markdown), device, host-buffer and file paths")
    ap.add_argument("--max-log2", type=int, default=20)
    ap.add_argument("--sets", default="1,2,4,8,16")
    ap.add_argument("--fig3-events", type=int, default=131072)
    ap.add_argument("--parity-report", action="store_true", help="error statistics against tests/golden/full_cfg*.npz (markdown)")
    args = ap.parse_args()
    if args.sweep:
        run_sweep(args)
        return
    if args.parity_report:
        run_parity_report(args)
        return
    args.config = args.config or 5
    if args.impl == "reference":
        run_reference(args)
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_2312_07440_b200 import binding as B, microbench as MB

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the reweighting path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c = ev.config(args.config)
    n = args.events or c.n_events
    dtype = "f64" if args.precision == "fp64" else "f32"
    flush_buf = torch.zeros(64 * 1024 * 1024, dtype=torch.float64, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    barrier()
    with ClockSampler(local) as cs:
        barrier()
        # --events beyond 2^20: the seeded set of 2^20 events tiled (the asymptotic size of the launch-bound cfg 1)
        res = time_config(torch, B, c, args.precision, n, args.steps, args.warmup, rank, flush_buf, tile_from=(1 << 20) if n > (1 << 20) else 0)
        barrier()
    clocks = cs.summary()
    total_s = max_over_ranks(sum(res["ms"]) * 1e-3)
    value = sharding.aggregate_throughput([n] * world, args.steps, total_s)      # all ranks' events over the slowest rank's time
    ms_per_step = total_s * 1e3 / args.steps

    # ---- e2e: the C-ABI call a user makes with HOST buffers (pinned), copies inside the timed region ----
    m, w = res["host"]
    pm, pw = torch.from_numpy(m).pin_memory(), torch.from_numpy(w).pin_memory()
    po = torch.empty((3, n), dtype=torch.float64).pin_memory()
    hm, hw, ho = pm.numpy(), pw.numpy(), po.numpy()
    st = torch.cuda.current_stream().cuda_stream
    for _ in range(2):
        B.rwgt_run_host(res["rw"].h, hm, hw, ho[0], ho[1], ho[2], st)
    barrier()
    t0 = time.perf_counter()
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(e2e_steps):
        B.rwgt_run_host(res["rw"].h, hm, hw, ho[0], ho[1], ho[2], st)     # synchronises the stream itself
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    e2e_val = sharding.aggregate_throughput([n] * world, e2e_steps, e2e_s)
    same = bool(np.array_equal(ho, res["out"].cpu().numpy()))

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the (single) kernel of a step: the FP64 (FP32) arithmetic pipe ----
    # FP64 mode: DFMA and DMMA share one pipe on B200 (include/rwgt_microbench.h kind 7), so the numerator is the vector flops
    # plus the algorithmic flops of the colour form (a5, run as mma.m8n8k4).  FP32/mixed: the vector flops against the
    # FP32 pipe; the colour form stays on the FP64 pipe and is reported beside it.
    peaks = measured_peaks()
    kernel_ms = statistics.mean(res["ms"])
    vec_flops, col_flops = res["flops_per_event"] * n, res["tensor_flops_per_event"] * n
    flops = vec_flops + (col_flops if dtype == "f64" else 0.0)
    achieved_tf = flops / (kernel_ms * 1e-3) / 1e12
    max_mhz = clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
    peak_tf = alu_peak_tflops(dtype, max_mhz)
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    traffic, traffic_build, ncu_fpe = None, None, None
    try:
        counts = json.load(open(os.path.join(ROOT, "profiles", "counts.json")))
        ent = counts[f"cfg{c.index}_{args.precision}"]
        # the ncu figures describe ONE build of the library: they are reported only when the loaded library is that build
        if n == c.n_events and ent.get("library_build_id") == B.rwgt_build_id():
            traffic, traffic_build = ent["traffic_bytes"], ent["library_build_id"]
            if dtype == "f64" and ent.get("fp64_vector_flops_per_launch_ncu"):
                ncu_fpe = ent["fp64_vector_flops_per_launch_ncu"] / n      # executed DFMA x 2 + DMUL + DADD per event, same capture
    except Exception:
        pass
    micro = {}
    kinds = ({"fma_chain": 0, "fma_3_distinct_sources": 3, "fma_1_reused_source": 4, "dmma_chain": 2, "dfma_and_dmma_concurrent": 7}
             if dtype == "f64" else {"fma_chain": 1, "fma_3_distinct_sources": 5, "fma_1_reused_source": 6,
                            "ffma2_chain": 8, "ffma2_3_distinct_sources": 9, "ffma2_1_reused_source": 10})
    for name, kind in kinds.items():
        try:
            micro[name] = MB.rwgt_microbench_peak(kind)     # register-resident microbenchmarks, same session
        except Exception:
            micro[name] = None
    chain_tf = micro.get("fma_chain")
    roofline = {"bound": "alu", "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved_tf / peak_tf, "traffic": traffic,
                "traffic_source": (f"ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, profiles/counts.json, measured on build {traffic_build}") if traffic else None,
                "peak_source": f"derived: 148 SM x {FP64_LANES_PER_SM if dtype == 'f64' else FP32_LANES_PER_SM} FMA lanes x 2 flop x {max_mhz:g} MHz (max SM clock); DESIGN.md Roofline",
                "peak_fma_chain_measured": chain_tf, "frac_of_fma_chain_measured": (achieved_tf / chain_tf) if chain_tf else None,
                "microbench_tflops": micro,
                "frac_at_clock_under_load": (achieved_tf / alu_peak_tflops(dtype, clocks["sm_mhz"])) if clocks.get("sm_mhz") else None,
                "flops_per_event": res["flops_per_event"] + (res["tensor_flops_per_event"] if dtype == "f64" else 0.0),
                "flops_per_event_kind": "algorithmic operation count of the schedule (include/rwgt.h rwgt_flops_per_event); FP32/mixed: model only, FFMA2 is not in ncu's FFMA counters",
                "vector_flops_per_event": res["flops_per_event"], "colour_form_flops_per_event": res["tensor_flops_per_event"],
                "vector_flops_per_event_ncu": ncu_fpe,
                "vector_flops_model_over_ncu": (res["flops_per_event"] / ncu_fpe) if ncu_fpe else None,
                "kernel_ms": kernel_ms,
                "colour_form_fp64": {"flops_per_event": res["tensor_flops_per_event"],
                                     "achieved_tflops": col_flops / (kernel_ms * 1e-3) / 1e12,
                                     "note": "mma.m8n8k4 on the FP64 pipe (shared with DFMA); included in `achieved` in FP64 mode only"},
                "hbm": {"achieved_gbs": bytes_per_event(c) * n / (kernel_ms * 1e-3) / 1e9, "peak_gbs": hbm_peak,
                        "peak_source": "MEASURED_PEAKS.json" if peaks.get("hbm_gbs") else "fallback"}}
    roofline["hbm"]["frac"] = roofline["hbm"]["achieved_gbs"] / roofline["hbm"]["peak_gbs"]

    line = {"metric": "reweighted events/s (both |M|^2)", "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": dtype, "data": "synthetic",
            "config": {"workload": workload_name(c, n), "events_per_gpu": n, "precision": args.precision, "l2": res["l2"],
                       "seed": c.seed, "kappa": 0.1 if 1 < c.index < 6 else None},
            "clocks": clocks, "gpu_launches": args.steps,
            "e2e": {"value": e2e_val, "unit": "events/s", "h2d_bytes_per_step": int(m.nbytes + w.nbytes), "d2h_bytes_per_step": int(3 * n * 8),
                    "steps": e2e_steps, "matches_device_path": same},
            "roofline": roofline}

    # ---- cpu_baseline: the oracle on a bounded sample of the same workload (rank 0, N = 1 only) ----
    if world == 1 and not args.no_cpu_baseline:
        import oracle as orc
        cores = os.cpu_count() or 1
        ns = min(n, max(8, int(ORACLE_PER_CORE[c.index] * cores * 12.0)))
        t0 = time.perf_counter()
        a, b, wn, used = orc.reweight(c.process, c.params_old, c.params_new, m[:, :, :ns].copy(), w[:ns].copy())
        dt = time.perf_counter() - t0
        gpu = res["out"][:, :ns].cpu().numpy()
        err = max(float(np.abs(gpu[0] / a - 1).max()), float(np.abs(gpu[1] / b - 1).max()), float(np.abs(gpu[2] / wn - 1).max()))
        line["cpu_baseline"] = {"value": ns / dt, "unit": "events/s", "cores": used, "kind": "oracle",
                                "sample": f"first {ns} events of the same seeded set, both parameter sets, {dt:.1f} s",
                                "max_rel_err_gpu_vs_oracle_on_sample": err}

    # ---- every config / precision with the same --steps / --warmup (north_star targets: cfgs 4, 5 FMA fraction, cfg 1 HBM) ----
    if world == 1 and not args.no_extra:
        per_config = [per_config_entry(c, args.precision, dict(res, n=n), max_mhz, hbm_peak)]
        extra = []
        for cc in ev.CONFIGS:
            for prec in cc.precisions + (("mixed",) if "fp32" in cc.precisions else ()):
                if cc.index == c.index and prec == args.precision:
                    continue
                try:
                    rr = time_config(torch, B, cc, prec, cc.n_events, args.steps, args.warmup, 0, flush_buf)
                    rr["n"] = cc.n_events
                    per_config.append(per_config_entry(cc, prec, rr, max_mhz, hbm_peak))
                    rr["rw"].close()
                except Exception as ex:  # keep the headline line alive
                    per_config.append({"cfg": cc.index, "precision": prec, "error": str(ex)})
        # cfg 1 is launch-latency-bound at its 16,384 events: the same distribution at n = 2^24 (buffers >> L2)
        try:
            c1 = ev.config(1)
            rr = time_config(torch, B, c1, "fp64", 1 << 24, args.steps, args.warmup, 0, flush_buf, tile_from=1 << 20)
            rr["n"] = 1 << 24
            e1 = per_config_entry(c1, "fp64", rr, max_mhz, hbm_peak)
            e1["note"] = "asymptotic size: the seeded set of 2^20 events tiled 16x (buffers >> L2)"
            per_config.append(e1)
            rr["rw"].close()
        except Exception as ex:
            per_config.append({"cfg": 1, "n": 1 << 24, "error": str(ex)})
        per_config.sort(key=lambda e: (e.get("cfg", 0), e.get("precision", ""), e.get("n", 0)))
        roofline["per_config"] = per_config
        # K new parameter sets in one pass (PAPER.md:87 step 7, Fig. 3 axis).  bench<K>: kappa = 0.1 (k+1) / K on both
        # gluon self-couplings (the polynomial mode's best case at n >= 4: rank n-1..n); general4: independent ggg / gggg scales and another
        # alpha_s (higher rank: the generic case); every line is compared with the oracle values stored for its list on the multi-round sample
        # of the SAME launch (tests/golden/ksets_*.npz, written by the oracle alone), the old set with every event of full_cfg<N>.npz
        for ci, lname in ((2, "bench8"), (3, "bench8"), (4, "bench8"), (4, "general4"), (5, "bench4"), (5, "bench16"), (5, "general4")):
            try:
                cc = ev.config(ci)
                sets = ev.kset_list(cc, lname)
                K = len(sets)
                rr = time_config(torch, B, cc, "fp64", cc.n_events, max(3, args.steps // 4), 3, 0, flush_buf, new_sets=sets)
                kms = statistics.mean(rr["ms"])
                kline = {"workload": workload_name(cc, cc.n_events) + f" with K={K} new parameter sets in one pass (list {lname})", "precision": "fp64",
                        "events_per_s": cc.n_events / (kms * 1e-3), "new_weights_per_s": K * cc.n_events / (kms * 1e-3), "kernel_ms": kms, "l2": rr["l2"]}
                gfile = os.path.join(ROOT, "tests", "golden", f"ksets_cfg{ci}_{lname}.npz")
                if os.path.exists(gfile):
                    g = np.load(gfile)
                    got = rr["out"].cpu().numpy()
                    sel = g["idx"]
                    err = max(np.abs(got[1:1 + K, sel] / g["me_new"] - 1).max(), np.abs(got[1 + K:, sel] / g["w_new"] - 1).max(), np.abs(got[0, sel] / g["me_old"] - 1).max())
                    kline["max_rel_err_vs_golden"] = float(err)
                    kline["golden_events"] = int(len(sel))
                extra.append(kline)
                rr["rw"].close()
            except Exception as ex:
                extra.append({"workload": f"cfg{ci} {lname}", "error": str(ex)})
        # cfg 1 at its stated 16,384 events is launch-latency-bound: the same launch captured in a CUDA graph (20 launches per replay)
        try:
            c1 = ev.config(1)
            m1, w1 = ev.generate(c1)
            dm1, dw1 = torch.from_numpy(m1).cuda(), torch.from_numpy(w1).cuda()
            r1 = B.Reweighter(c1.process, c1.params_old, c1.params_new, "fp64")
            o1 = torch.empty((3, c1.n_events), dtype=torch.float64, device="cuda")
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                r1.run(dm1, dw1, o1)
            torch.cuda.current_stream().wait_stream(side)
            g = torch.cuda.CUDAGraph()
            reps = 20
            with torch.cuda.graph(g):
                for _ in range(reps):
                    r1.run(dm1, dw1, o1)
            ts = []
            for it in range(3 + 10):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                g.replay()
                e1.record()
                torch.cuda.synchronize()
                if it >= 3:
                    ts.append(e0.elapsed_time(e1) / reps)
            kms = statistics.mean(ts)
            extra.append({"workload": workload_name(c1, c1.n_events) + f" replayed from a CUDA graph of {reps} launches (inputs stay in L2)", "precision": "fp64",
                          "events_per_s": c1.n_events / (kms * 1e-3), "kernel_ms": kms, "l2": "not flushed (graph replay)"})
            r1.close()
        except Exception as ex:
            extra.append({"workload": "epem_mupmum CUDA graph", "error": str(ex)})
        line["other_configs"] = extra
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
