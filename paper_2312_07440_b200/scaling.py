"""The paper's two experiments on its own process e+ e- -> 5 gamma (Table 1; Fig. 2: runtime
against the number of events for one parameter set; Fig. 3: runtime against the number of parameter sets), run
through this library on one GPU.  As in the paper every point is the mean of 5 runs with its min/max.

    python -m paper_2312_07440_b200.scaling [--config 6] [--max-log2 20] [--sets 1,2,4,8,16] [--fig3-events 131072]

Columns: device = rwgt_run_multi on device-resident buffers (CUDA events); host = rwgt_run_multi_host on pinned host buffers,
host<->device copies inside the timed call (the transfer overhead the paper describes for small n).
Each parameter set draws its electroweak coupling at random.  Prints a markdown table (profiles/r1_scaling_5gamma.md)."""
import argparse
import time

import numpy as np


def stats(ts):
    return f"{np.mean(ts):.4f} ({min(ts):.4f}-{max(ts):.4f})"


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--max-log2", type=int, default=20)
    ap.add_argument("--sets", default="1,2,4,8,16")
    ap.add_argument("--fig3-events", type=int, default=131072)
    ap.add_argument("--config", type=int, default=6, help="6 = the paper's process; 1..5 = the BASELINE.json configs (SURVEY 8(d) D3 sweep)")
    args = ap.parse_args()
    import torch
    from . import binding as B, events as ev
    c = ev.config(args.config)
    nmax = max(1 << args.max_log2, args.fig3_events)
    m0, w0 = ev.generate(c, min(nmax, c.n_events))
    reps = (nmax + m0.shape[2] - 1) // m0.shape[2]
    m = np.tile(m0, (1, 1, reps))[:, :, :nmax].copy()
    w = np.tile(w0, reps)[:nmax].copy()
    rng = np.random.default_rng(c.seed)

    def new_sets(k):
        if c.index == 6:      # a random electroweak coupling per set
            return [ev.params(alpha_em=float(a)) for a in rng.uniform(0.5, 2.0, size=k) / 132.5]
        if c.index == 1:
            return [ev.params(GammaZ=float(g), sin2_thetaW=float(x)) for g, x in zip(rng.uniform(2.3, 2.7, size=k), rng.uniform(0.22, 0.24, size=k))]
        return [ev.params(ggg_scale=float(1 + x), gggg_scale=float(1 + x)) for x in rng.uniform(-0.2, 0.2, size=k)]

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
        dev, host = [], []
        for it in range(2 + 5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            B.rwgt_run_multi(h, dm.data_ptr(), dw.data_ptr(), a.data_ptr(), b.data_ptr(), o.data_ptr(), n, st)
            e1.record()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            B.rwgt_run_multi_host(h, mh.numpy(), wh.numpy(), ha.numpy(), hb.numpy(), ho.numpy())
            t1 = time.perf_counter()
            if it >= 2:
                dev.append(e0.elapsed_time(e1))
                host.append((t1 - t0) * 1e3)
        assert np.array_equal(ho.numpy(), o.cpu().numpy())
        B.rwgt_destroy(h)
        return dev, host

    print(f"# {c.process} (config {c.index}), FP64\n")
    print("## Runtime against the number of events, one parameter set (PAPER.md:105 Fig. 2), ms: mean (min-max) of 5\n")
    print("| events | device ms | host-buffer ms | device events/s | host-buffer events/s |\n|---|---|---|---|---|")
    for lg in range(0, args.max_log2 + 1, 2):
        n = 1 << lg
        dev, host = measure(n, 1)
        print(f"| {n} | {stats(dev)} | {stats(host)} | {n / np.mean(dev) * 1e3:.3e} | {n / np.mean(host) * 1e3:.3e} |", flush=True)
    n = args.fig3_events
    print(f"\n## Runtime against the number of parameter sets, {n} events (PAPER.md:117 Fig. 3), ms: mean (min-max) of 5\n")
    print("| parameter sets | device ms | host-buffer ms | new weights/s (device) |\n|---|---|---|---|")
    for K in [int(x) for x in args.sets.split(",")]:
        dev, host = measure(n, K)
        print(f"| {K} | {stats(dev)} | {stats(host)} | {K * n / np.mean(dev) * 1e3:.3e} |", flush=True)


if __name__ == "__main__":
    main()
