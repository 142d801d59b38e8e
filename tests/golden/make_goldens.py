#!/usr/bin/env python
"""Writes the full-set expected values tests/golden/full_cfg<N>.npz: |M|^2, |M'|^2 and W' of the first n events of the
seeded set of config N (paper_2312_07440_b200/events.py), computed by the CPU oracle and by nothing else.

    python tests/golden/make_goldens.py --config 2 [--events 1048576] [--threads 6] [--chunk 4096]

Calls only oracle/ (the arithmetic) and events.py (the seeded inputs, which hold none of the method's arithmetic).  It never
imports or loads the CUDA path.  The event sets are prefix-stable (the first n accepted candidates in counter order), so a
later call with a larger --events extends an existing file: the events already stored are kept and only the new ones are
evaluated.  The GPU parity tests (tests/test_gpu_goldens.py) compare FP64, FP32 and mixed launches with these files element
by element, so no oracle time is spent on the GPU box.

    python tests/golden/make_goldens.py --config 5 --sets bench16 [--threads 8]

writes tests/golden/ksets_cfg<N>_<list>.npz instead: for the named list of K new parameter sets (events.kset_list: what bench.py
times with K > 1, lists with other top masses, independent coupling scales) the oracle's |M|^2, |M'_k|^2 and W'_k on the
events events.kset_sample picks from the config's FULL seeded set (a prefix longer than two rounds of the persistent launch,
a strided sample of every later round, the tail), one orc.reweight call per set.  tests/test_gpu_ksets.py launches the full
set and compares these events (VERDICT r2 item 1; PAPER.md:87 step 7, :117)."""
import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
import oracle as orc  # noqa: E402
from paper_2312_07440_b200 import events as ev  # noqa: E402

DEFAULT_EVENTS = {1: 16384, 2: 1048576, 3: 262144, 4: 32768, 5: 8192, 6: 32768}


def path(idx: int) -> str:
    return os.path.join(HERE, f"full_cfg{idx}.npz")


def kset_path(idx: int, name: str) -> str:
    return os.path.join(HERE, f"ksets_cfg{idx}_{name}.npz")


def make_ksets(c, name: str, threads: int) -> None:
    sets = ev.kset_list(c, name)
    idx = ev.kset_sample(c)
    m, w = ev.generate(c)
    ms, ws = np.ascontiguousarray(m[:, :, idx]), w[idx].copy()
    K = len(sets)
    me_old, me_new, w_new = np.full(len(idx), np.nan), np.full((K, len(idx)), np.nan), np.full((K, len(idx)), np.nan)
    t0 = time.time()
    for k, pn in enumerate(sets):
        a, b, wn, used = orc.reweight(c.process, c.params_old, pn, ms, ws, nthreads=threads)
        assert k == 0 or np.array_equal(a, me_old)
        me_old, me_new[k], w_new[k] = a, b, wn
        print(f"cfg {c.index} {name}: set {k + 1}/{K}, {len(idx)} events, {time.time() - t0:.0f} s, {used} threads", flush=True)
    np.savez(kset_path(c.index, name) + ".tmp.npz", idx=idx, sets=np.array(sets), me_old=me_old, me_new=me_new, w_new=w_new, seed=c.seed,
             process=c.process, params_old=c.params_old)
    os.replace(kset_path(c.index, name) + ".tmp.npz", kset_path(c.index, name))


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--events", type=int, default=0)
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--sets", default="", help="name of a K-set list (events.KSET_LISTS): write ksets_cfg<N>_<list>.npz")
    args = ap.parse_args()
    c = ev.config(args.config)
    if args.sets:
        make_ksets(c, args.sets, args.threads)
        return
    n = min(args.events or DEFAULT_EVENTS[c.index], c.n_events)
    out = np.full((3, n), np.nan)
    done = 0
    if os.path.exists(path(c.index)):
        old = np.load(path(c.index))
        assert int(old["seed"]) == c.seed and np.array_equal(old["params_old"], c.params_old) and np.array_equal(old["params_new"], c.params_new)
        done = min(n, old["out"].shape[1])
        out[:, :done] = old["out"][:, :done]
    m, w = ev.generate(c, n)
    chunk = args.chunk or max(64, n // 64)
    t0 = time.time()
    while done < n:
        hi = min(n, done + chunk)
        a, b, wn, used = orc.reweight(c.process, c.params_old, c.params_new, np.ascontiguousarray(m[:, :, done:hi]), w[done:hi].copy(), nthreads=args.threads)
        out[0, done:hi], out[1, done:hi], out[2, done:hi] = a, b, wn
        done = hi
        np.savez(path(c.index) + ".tmp.npz", out=out[:, :done], seed=c.seed, process=c.process, params_old=c.params_old, params_new=c.params_new)
        os.replace(path(c.index) + ".tmp.npz", path(c.index))
        print(f"cfg {c.index}: {done}/{n} events, {time.time() - t0:.0f} s, {used} threads", flush=True)


if __name__ == "__main__":
    main()
