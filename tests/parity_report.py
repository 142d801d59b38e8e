"""Parity report: per config and precision the max / median relative error of |M|^2, |M'|^2, W' of the CUDA path
against the CPU oracle on the first N events of the seeded set, the number of events over tolerance and the worst event.

    python tests/parity_report.py [--scale 1]        # needs a GPU; prints a markdown table (profiles/r1_parity.md)

Not collected by pytest (no test_ prefix); lives under tests/ because only tests/, smoke() and bench.py may use the oracle."""
import argparse
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import oracle as orc  # noqa: E402
from paper_2312_07440_b200 import binding as B, events as ev  # noqa: E402

N = {1: 65536, 2: 65536, 3: 8192, 4: 1024, 5: 96, 6: 512}
TOL = {"fp64": (1e-11, 1e-11), "fp32": (1e-4, 1e-6), "mixed": (1e-4, 1e-6)}


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--scale", type=float, default=1.0)
    args = ap.parse_args()
    import torch
    print("| cfg | process | precision | events | max rel. err | median rel. err | tolerance (max / median) | events over max tolerance | worst event | oracle threads |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for idx in (1, 2, 3, 4, 5, 6):
        c = ev.config(idx)
        n = max(8, int(N[idx] * args.scale))
        m, w = ev.generate(c, n)
        a, b, wn, used = orc.reweight(c.process, c.params_old, c.params_new, m, w)
        ref = np.stack([a, b, wn])
        dm, dw = torch.from_numpy(m).cuda(), torch.from_numpy(w).cuda()
        for prec in c.precisions + (("mixed",) if "fp32" in c.precisions else ()):
            r = B.Reweighter(c.process, c.params_old, c.params_new, prec)
            got = r.run(dm, dw).cpu().numpy()
            r.close()
            e = np.abs(got / ref - 1).max(axis=0)           # per event: worst of the three outputs
            tmax, tmed = TOL[prec]
            print(f"| {idx} | {c.process} | {prec} | {n} | {e.max():.2e} | {np.median(e):.2e} | {tmax:g} / {tmed:g} | {int((e > tmax).sum())} | {int(e.argmax())} | {used} |", flush=True)


if __name__ == "__main__":
    main()
