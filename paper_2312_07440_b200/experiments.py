"""Phase-removal timings of the ordered-current engine (diagnostic; results of the flagged runs are wrong by construction).

    python -m paper_2312_07440_b200.build --experiment      # librwgt_exp.so, compiled with -DRWGT_EXPERIMENT
    python -m paper_2312_07440_b200.experiments [--configs 4,5] [--precisions fp64,fp32]

RWGT_EXP bits: 1 = every table load reads entry 0 (conflict-free broadcast: removes shared-memory bandwidth and bank
conflicts, keeps the instruction stream), 2 = skip the colour mma, 4 = skip the current levels, 8 = skip the amplitude tasks.
Output feeds profiles/r1_experiments.md."""
import argparse
import os
import statistics

import numpy as np


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="4,5")
    ap.add_argument("--precisions", default="fp64,fp32")
    ap.add_argument("--flags", default="0,1,2,4,8,6,10")
    args = ap.parse_args()
    import torch
    from . import binding as B, build, events as ev
    if not os.path.exists(build.LIB_EXP):
        build.build(experiment=True)
    B.LIB_PATH = build.LIB_EXP
    for ci in [int(x) for x in args.configs.split(",")]:
        c = ev.config(ci)
        n = c.n_events
        m0, w0 = ev.generate(c, min(n, 4096))
        reps = (n + m0.shape[2] - 1) // m0.shape[2]
        m, w = np.tile(m0, (1, 1, reps))[:, :, :n].copy(), np.tile(w0, reps)[:n].copy()
        dm, dw = torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda()
        out = torch.empty((3, n), dtype=torch.float64, device="cuda")
        for prec in args.precisions.split(","):
            r = B.Reweighter(c.process, c.params_old, c.params_new, prec)
            for f in [int(x) for x in args.flags.split(",")]:
                os.environ["RWGT_EXP"] = str(f)
                for _ in range(2):
                    r.run(dm, dw, out)
                torch.cuda.synchronize()
                ts = []
                for _ in range(5):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    r.run(dm, dw, out)
                    e1.record()
                    torch.cuda.synchronize()
                    ts.append(e0.elapsed_time(e1))
                print(f"cfg{ci} {prec} n={n} RWGT_EXP={f}: {statistics.median(ts):.3f} ms", flush=True)
            r.close()


if __name__ == "__main__":
    main()
