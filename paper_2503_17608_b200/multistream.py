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
