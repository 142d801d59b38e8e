#!/usr/bin/env python
"""bench.py — reweighted events/s of the LO reweighting hot path (eq. 3; PAPER.md:87 steps 3-6).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--precision fp64] [--impl reference]

A step = one pass of the whole hot path (one rwgt_run launch: a1-a7 of SURVEY §8(a)) over the synthetic
event set of one BASELINE.json config (default configs[1] = gg -> ttbar, 1,048,576 events).  Prints ONE
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

from paper_2312_07440_b200 import events as ev  # noqa: E402

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
    per_core = {1: 25000.0, 2: 500.0, 3: 55.0, 4: 5.0, 5: 1.1, 6: 5.0}[c.index]       # rough oracle events/s/core, sizes the sample only
    cores = os.cpu_count() or 1
    n = args.ref_events or max(8, int(per_core * cores * 4.0))                    # ~4 s per step
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


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index 1..5 (default 2 = configs[1]); 6 = the paper's own e+e- -> 5 gamma (PAPER.md:72-77)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "mixed"])
    ap.add_argument("--events", type=int, default=0, help="override the config's event count")
    ap.add_argument("--ref-events", type=int, default=0, help="reference arm: events per step")
    ap.add_argument("--no-extra", action="store_true", help="skip the per-config summary of the other configs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
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
    value = world * n * args.steps / total_s
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
    e2e_val = world * n * e2e_steps / e2e_s
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
    traffic = None
    try:
        traffic = json.load(open(os.path.join(ROOT, "profiles", "r1_counts.json")))[f"cfg{c.index}_{args.precision}"]["traffic_bytes"]
        if n != c.n_events:
            traffic = None
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
                "peak_source": f"derived: 148 SM x {FP64_LANES_PER_SM if dtype == 'f64' else FP32_LANES_PER_SM} FMA lanes x 2 flop x {max_mhz:g} MHz (max SM clock); DESIGN.md Roofline",
                "peak_fma_chain_measured": chain_tf, "frac_of_fma_chain_measured": (achieved_tf / chain_tf) if chain_tf else None,
                "microbench_tflops": micro,
                "frac_at_clock_under_load": (achieved_tf / alu_peak_tflops(dtype, clocks["sm_mhz"])) if clocks.get("sm_mhz") else None,
                "flops_per_event": res["flops_per_event"] + (res["tensor_flops_per_event"] if dtype == "f64" else 0.0),
                "vector_flops_per_event": res["flops_per_event"], "colour_form_flops_per_event": res["tensor_flops_per_event"],
                "kernel_ms": kernel_ms,
                "colour_form_fp64": {"flops_per_event": res["tensor_flops_per_event"],
                                     "achieved_tflops": col_flops / (kernel_ms * 1e-3) / 1e12,
                                     "note": "mma.m8n8k4 on the FP64 pipe (shared with DFMA); included in `achieved` in FP64 mode only"},
                "hbm": {"achieved_gbs": bytes_per_event(c) * n / (kernel_ms * 1e-3) / 1e9, "peak_gbs": peaks.get("hbm_gbs", 6650.0),
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
        per_core = {1: 25000.0, 2: 500.0, 3: 55.0, 4: 5.0, 5: 1.1, 6: 5.0}[c.index]
        cores = os.cpu_count() or 1
        ns = min(n, max(8, int(per_core * cores * 12.0)))
        t0 = time.perf_counter()
        a, b, wn, used = orc.reweight(c.process, c.params_old, c.params_new, m[:, :, :ns].copy(), w[:ns].copy())
        dt = time.perf_counter() - t0
        gpu = res["out"][:, :ns].cpu().numpy()
        err = max(float(np.abs(gpu[0] / a - 1).max()), float(np.abs(gpu[1] / b - 1).max()), float(np.abs(gpu[2] / wn - 1).max()))
        line["cpu_baseline"] = {"value": ns / dt, "unit": "events/s", "cores": used, "kind": "oracle",
                                "sample": f"first {ns} events of the same seeded set, both parameter sets, {dt:.1f} s",
                                "max_rel_err_gpu_vs_oracle_on_sample": err}

    # ---- the other configs / precisions, short runs, same protocol (context for the north_star targets) ----
    if world == 1 and not args.no_extra:
        extra = []
        for cc in ev.CONFIGS:
            for prec in cc.precisions:
                if cc.index == c.index and prec == args.precision:
                    continue
                try:
                    rr = time_config(torch, B, cc, prec, cc.n_events, 5, 3, 0, flush_buf)
                    kms = statistics.mean(rr["ms"])
                    dt_ = "f64" if prec == "fp64" else "f32"
                    fpe = rr["flops_per_event"] + (rr["tensor_flops_per_event"] if dt_ == "f64" else 0.0)
                    tf = fpe * cc.n_events / (kms * 1e-3) / 1e12
                    extra.append({"workload": workload_name(cc, cc.n_events), "precision": prec, "events_per_s": cc.n_events / (kms * 1e-3),
                                  "kernel_ms": kms, "alu_tflops": tf, "alu_frac": tf / alu_peak_tflops(dt_, max_mhz),
                                  "hbm_gbs": bytes_per_event(cc) * cc.n_events / (kms * 1e-3) / 1e9,
                                  "hbm_frac": bytes_per_event(cc) * cc.n_events / (kms * 1e-3) / 1e9 / roofline["hbm"]["peak_gbs"], "l2": rr["l2"]})
                    rr["rw"].close()
                except Exception as ex:  # keep the headline line alive
                    extra.append({"workload": workload_name(cc, cc.n_events), "precision": prec, "error": str(ex)})
        # K new parameter sets in one pass (PAPER.md:87 step 7, Fig. 3 axis): kappa = 0.1 k / K
        for ci, K in ((2, 8), (4, 8), (5, 4)):
            try:
                cc = ev.config(ci)
                sets = [ev.params(ggg_scale=1 + 0.1 * (k + 1) / K, gggg_scale=1 + 0.1 * (k + 1) / K) for k in range(K)]
                rr = time_config(torch, B, cc, "fp64", cc.n_events, 5, 3, 0, flush_buf, new_sets=sets)
                kms = statistics.mean(rr["ms"])
                fpe = rr["flops_per_event"] + rr["tensor_flops_per_event"]
                tf = fpe * cc.n_events / (kms * 1e-3) / 1e12
                extra.append({"workload": workload_name(cc, cc.n_events) + f" with K={K} new parameter sets in one pass", "precision": "fp64",
                              "events_per_s": cc.n_events / (kms * 1e-3), "new_weights_per_s": K * cc.n_events / (kms * 1e-3), "kernel_ms": kms,
                              "alu_tflops": tf, "alu_frac": tf / alu_peak_tflops("f64", max_mhz), "l2": rr["l2"]})
                rr["rw"].close()
            except Exception as ex:
                extra.append({"workload": f"cfg{ci} K={K}", "error": str(ex)})
        # cfg 1 is launch-latency-bound at its 16,384 events: the same distribution at n = 2^24 (buffers >> L2)
        try:
            c1 = ev.config(1)
            rr = time_config(torch, B, c1, "fp64", 1 << 24, 5, 3, 0, flush_buf, tile_from=1 << 20)
            kms = statistics.mean(rr["ms"]); n1 = 1 << 24
            gbs = bytes_per_event(c1) * n1 / (kms * 1e-3) / 1e9
            tf = rr["flops_per_event"] * n1 / (kms * 1e-3) / 1e12
            extra.append({"workload": workload_name(c1, n1) + " (asymptotic: the seeded set of 2^20 events tiled 16x)", "precision": "fp64",
                          "events_per_s": n1 / (kms * 1e-3), "kernel_ms": kms, "alu_tflops": tf, "alu_frac": tf / alu_peak_tflops("f64", max_mhz),
                          "hbm_gbs": gbs, "hbm_frac": gbs / roofline["hbm"]["peak_gbs"], "l2": rr["l2"]})
            rr["rw"].close()
        except Exception as ex:
            extra.append({"workload": "epem_mupmum n=2^24", "error": str(ex)})
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
