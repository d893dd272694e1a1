"""Counter / slice trace export (fig. 2: per-iteration active and queued tracks and
per-action kernel time, which the paper takes from Perfetto).

The library stamps every kernel of every iteration with the GPU's global nanosecond timer (include/cel.h: cel_trace,
option "trace"); this module turns the stamps and the per-iteration action counts into Chrome-trace JSON, which the
Perfetto UI (ui.perfetto.dev) and chrome://tracing read — no SDK. Formatting only: nothing of the method is computed here.

    python -m paper_2503_17608_b200.trace_export --workload config2 --out gpurun_out/trace.json

prints a per-iteration table (kernel start + duration in us) and writes the JSON.
"""
import argparse
import json

import numpy as np

ACTIONS = ("PE", "PAIR", "COMPTON", "MOVE_G", "MOVE_C", "BREMS", "ANNIH", "VACANT")
NEVER = np.iinfo(np.uint64).max


def chrome_trace(names, stamps, counts, label="celstep"):
    """names: kernel names; stamps: [n_iter][n_kernels][2] uint64 ns (start, end; {UINT64_MAX, 0} = did not run);
    counts: [n_iter][8] action counts after P1. Returns the Chrome-trace dict."""
    stamps = np.asarray(stamps, dtype=np.uint64)
    ran = (stamps[:, :, 1] > 0) & (stamps[:, :, 0] != NEVER)
    if not ran.any():
        return {"traceEvents": [], "displayTimeUnit": "ns"}
    t0 = int(stamps[:, :, 0][ran].min())
    ev = [{"name": "process_name", "ph": "M", "pid": 0, "args": {"name": label}}]
    for j, n in enumerate(names):
        ev.append({"name": "thread_name", "ph": "M", "pid": 0, "tid": j, "args": {"name": n}})
    n_iter = min(len(stamps), len(counts)) if counts is not None and len(counts) else len(stamps)
    for k in range(n_iter):
        for j, n in enumerate(names):
            if not ran[k, j]:
                continue
            s, e = int(stamps[k, j, 0]), int(stamps[k, j, 1])
            ev.append({"name": n, "cat": "kernel", "ph": "X", "pid": 0, "tid": j, "ts": (s - t0) / 1e3,
                       "dur": max(e - s, 0) / 1e3, "args": {"iteration": k}})
        if counts is not None and len(counts) > k and ran[k].any():
            ts = (int(stamps[k, :, 0][ran[k]].min()) - t0) / 1e3
            c = [int(x) for x in counts[k]]
            ev.append({"name": "tracks", "ph": "C", "pid": 0, "ts": ts, "args": {"alive": sum(c[:7])}})
            ev.append({"name": "actions", "ph": "C", "pid": 0, "ts": ts, "args": {a: c[i] for i, a in enumerate(ACTIONS[:7])}})
    return {"traceEvents": ev, "displayTimeUnit": "ns"}


def summary_rows(names, stamps, counts, every=20):
    """text table: iteration, live tracks, per kernel `start+duration` in us relative to the iteration's first kernel"""
    stamps = np.asarray(stamps, dtype=np.uint64).astype(np.int64)
    n = min(len(stamps), len(counts))
    used = [j for j in range(len(names)) if (stamps[:n, j, 1] > 0).any()]
    rows = ["iter   alive | " + " | ".join(f"{names[j]:>13s}" for j in used) + " | length"]
    for k in range(n):
        if not (k % every == 0 or k >= n - 3):
            continue
        ok = [j for j in used if stamps[k, j, 1] > 0]
        if not ok:
            continue
        base = min(stamps[k, j, 0] for j in ok)
        end = max(stamps[k, j, 1] for j in ok)
        cells = []
        for j in used:
            s, e = stamps[k, j]
            cells.append(f"{(s - base) / 1e3:6.1f}+{(e - s) / 1e3:6.1f}" if e > 0 else " " * 13)
        rows.append(f"{k:4d} {int(sum(counts[k][:7])):7d} | " + " | ".join(cells) + f" | {(end - base) / 1e3:6.1f}")
    return rows


def main():
    import torch
    from . import binding, workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="config2", choices=["config1", "config2", "config3", "config4", "config5"])
    ap.add_argument("--events", type=int, default=0)
    ap.add_argument("--slots", type=int, default=0)
    ap.add_argument("--sort-mode", type=int, default=1, choices=[0, 1, 2, 3])
    ap.add_argument("--iters", type=int, default=512, help="iterations to stamp")
    ap.add_argument("--out", default="trace.json")
    args = ap.parse_args()
    assert torch.cuda.is_available(), "trace_export needs a CUDA device"
    torch.cuda.set_device(0)
    kw = {k: v for k, v in (("n_events", args.events), ("n_slots", args.slots)) if v}
    w = getattr(W, args.workload)(sort_mode=args.sort_mode, **kw)
    ctx = binding.from_workload(w)
    ctx.transport(w.primaries, w.n_events); ctx.tallies_view()          # warm-up
    ctx.set_option("trace", args.iters)
    ctx.transport(w.primaries, w.n_events)
    v = ctx.tallies_view()
    names, stamps = ctx.trace()
    counts = ctx.counts()
    with open(args.out, "w") as f:
        json.dump(chrome_trace(names, stamps, counts, label=f"{w.name} sort {args.sort_mode}"), f)
    print(f"{w.name}: {v['iterations']} iterations, {v['track_steps']} track-steps, {v['seconds'] * 1e3:.2f} ms traced "
          f"(the stamps cost two integer atomics per block and kernel) -> {args.out}")
    print("\n".join(summary_rows(names, stamps, counts)))
    ctx.close()


if __name__ == "__main__":
    main()
