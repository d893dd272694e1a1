"""Event-parallel multi-stream execution on ONE GPU (section 3.4).

The paper's Geant4-integrated application gives every CPU thread its own CUDA stream and its own track array, and
found that nothing may synchronise device-wide for this to pay. Here the same idea is applied to the
standalone model: the workload's events are split into K contiguous blocks (sharding.event_block), each block is
transported by its own cel_ctx with n_slots / K slots on its own non-blocking stream, driven by its own host thread
(ctypes releases the GIL during the C call; a context is used by one thread at a time, as include/cel.h requires).
The contexts share nothing, so the result of a block is bit-identical to transporting that block alone; what is
gained is that one context's latency-bound bookkeeping overlaps another context's action kernels.
Marshalling and threading only: every step of the path runs in the kernels of libcelstep.so.
"""
import threading

import numpy as np

from . import binding, sharding


class MultiStream:
    def __init__(self, workload, n_streams, sort_mode=None, options=None):
        self.w = workload
        self.k = int(n_streams)
        assert self.k >= 1 and workload.n_slots % self.k == 0
        self.parts = []
        for i in range(self.k):
            prim, n_local, lo = sharding.shard_primaries(workload.primaries, workload.n_events, i, self.k)
            ctx = binding.from_workload(workload, n_slots=workload.n_slots // self.k, sort_mode=sort_mode)
            for name, value in (options or {}).items():
                ctx.set_option(name, value)
            self.parts.append((ctx, prim, n_local, lo))

    def transport(self):
        """transport every block concurrently; returns when all of them have ended"""
        errors = []

        def run(ctx, prim, n_local):
            try:
                if n_local:
                    ctx.transport(prim, n_local)
            except Exception as e:   # surfaced to the caller below
                errors.append(e)

        threads = [threading.Thread(target=run, args=(c, p, n)) for c, p, n, _ in self.parts]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        if errors:
            raise errors[0]

    def views(self):
        return [c.tallies_view() if n else None for c, _, n, _ in self.parts]

    def tallies_fixed(self):
        """[n_events][n_bins+1] uint64, the blocks' tallies in event order"""
        rows = [v["fixed"] for v in self.views() if v is not None]
        return np.concatenate(rows, axis=0)

    def counters(self):
        vs = [v for v in self.views() if v is not None]
        return dict(track_steps=sum(v["track_steps"] for v in vs), secondaries=sum(v["secondaries"] for v in vs),
                    iterations=max(v["iterations"] for v in vs), kernel_launches=sum(v["kernel_launches"] for v in vs))

    def close(self):
        for c, _, _, _ in self.parts:
            c.close()
        self.parts = []


def main():
    """measurement of PAPER.md section 3.4 on one GPU: K event-parallel contexts, with the hit transfer off, stream-ordered
    (hits = 1) and synchronous (hits = 2, the paper's "before"); wall clock of the whole transport, best of `--repeat`"""
    import argparse
    import time
    import torch
    from . import workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="config2", choices=["config2", "config3", "config4", "config5"])
    ap.add_argument("--streams", default="1,2,4,8,16")
    ap.add_argument("--hits", default="0,1,2")
    ap.add_argument("--sort-mode", type=int, default=1)
    ap.add_argument("--repeat", type=int, default=3)
    args = ap.parse_args()
    assert torch.cuda.is_available(), "needs a CUDA device"
    w = getattr(W, args.workload)(sort_mode=args.sort_mode)
    print(f"# {w.name}: {w.n_events} events, {w.n_slots} slots in total, sort mode {args.sort_mode}; ms per transport (wall clock, best of {args.repeat})")
    print("# streams | " + " | ".join(f"hits={h}" for h in args.hits.split(",")) + " | hit records, MB to the host")
    for k in [int(x) for x in args.streams.split(",")]:
        cells, info = [], ""
        for h in [int(x) for x in args.hits.split(",")]:
            opts = {"hits": h, "hit_capacity": max(1 << 20, 16 * (w.n_slots // k))} if h else {}
            ms = MultiStream(w, k, options=opts)
            ms.transport()                                      # warm-up (graph capture, pinned allocations)
            best = 1e30
            for _ in range(args.repeat):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                ms.transport()
                if h:
                    hv = [c.hits_view() for c, _, n, _ in ms.parts if n]     # waits for the consumers
                else:
                    ms.views()
                best = min(best, time.perf_counter() - t0)
            if h:
                info = f"{sum(v['n_hits'] for v in hv)} records, {sum(v['bytes_d2h'] for v in hv) / 1e6:.0f} MB"
            cells.append(f"{best * 1e3:8.2f}")
            ms.close()
        print(f"{k:9d} | " + " | ".join(cells) + " | " + info, flush=True)


if __name__ == "__main__":
    main()
