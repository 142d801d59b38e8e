"""Reweight a binary event file from the command line: the paper's 8-step procedure end to end.

    python -m paper_2312_07440_b200.reweight_file events.rwgt results.rwgt --process gg_ttxg --new ggg_scale=1.1,gggg_scale=1.1 [--new ...]
    torchrun --nproc-per-node N -m paper_2312_07440_b200.reweight_file ...     # one rank per GPU, rank r writes results.rwgt.r

Events are independent: rank r of N takes the contiguous range sharding.shard_bounds(n, r, N) and writes its own result
file; there is no exchange step.  Everything on the path runs inside librwgt.so (rwgt_run_file); this module only parses arguments."""
import argparse
import os

from . import binding as B, events as ev, sharding


def parse_set(text: str):
    kw = {}
    for item in filter(None, text.split(",")):
        k, v = item.split("=")
        if k not in ev.PARAM_NAMES:
            raise SystemExit(f"unknown parameter {k!r}; known: {', '.join(ev.PARAM_NAMES)}")
        kw[k] = float(v)
    return ev.params(**kw)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("events")
    ap.add_argument("results")
    ap.add_argument("--process", default="", help="default: the process named in the event file")
    ap.add_argument("--old", default="", help="original parameter set, name=value,... (defaults: events.params())")
    ap.add_argument("--new", action="append", required=True, help="one new parameter set per --new")
    ap.add_argument("--precision", default="fp64", choices=list(B.PRECISIONS))
    args = ap.parse_args()
    import torch
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    process = args.process or B.event_file_process(args.events)
    n = B.event_file_n_events(args.events)
    lo, hi = sharding.shard_bounds(n, rank, world)
    h = B.rwgt_create_multi(process, parse_set(args.old), [parse_set(t) for t in args.new])
    B.rwgt_set_precision(h, args.precision)
    out = args.results if world == 1 else f"{args.results}.{rank}"
    B.rwgt_run_file(h, args.events, out, lo, hi - lo)
    B.rwgt_destroy(h)
    res = B.read_result_file(out)
    print(f"rank {rank}: events [{lo}, {hi}) -> {out}; sum W = {res['sum_w_old']:.12g}; sum W'_k = {', '.join(f'{x:.12g}' for x in res['sum_w_new'])}")


if __name__ == "__main__":
    main()
