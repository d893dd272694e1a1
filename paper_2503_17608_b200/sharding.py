"""Event sharding over ranks — host logic only, no arithmetic of the method.

Particle histories of different events are independent, and the tally is per event x bin, so the
path shards over events with no data-path collective: rank r transports the contiguous block of events
[lo_r, hi_r) in its own context. The only communication is the final exchange of the integer tallies
(an all_gather of uint64 rows; exact) and the max over ranks of the device time.
Works with any torch.distributed backend (nccl on GPUs; gloo in the CPU tests).
"""
import numpy as np
import torch
import torch.distributed as dist


def event_block(n_events: int, rank: int, world: int):
    """contiguous block [lo, hi) of event ids owned by `rank`; blocks differ in size by at most one event"""
    base, extra = divmod(int(n_events), int(world))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_primaries(primaries: np.ndarray, n_events: int, rank: int, world: int):
    """the primaries of this rank's events, with event ids renumbered from 0; returns (primaries, n_local_events, lo)"""
    lo, hi = event_block(n_events, rank, world)
    sel = (primaries["event"] >= lo) & (primaries["event"] < hi)
    local = primaries[sel].copy()
    local["event"] -= np.uint32(lo)
    return local, hi - lo, lo


def merge_tallies(local_fixed: np.ndarray, n_events: int, group=None, device="cpu") -> np.ndarray:
    """all_gather of the ranks' [n_local][n_bins+1] uint64 tallies into the global [n_events][n_bins+1] array
    (every rank gets it). Rows are padded to the largest block so that all_gather sees equal shapes."""
    world = dist.get_world_size(group)
    width = int(local_fixed.shape[1])
    rows = max(event_block(n_events, r, world)[1] - event_block(n_events, r, world)[0] for r in range(world))
    buf = np.zeros((rows, width), dtype=np.int64)
    buf[:local_fixed.shape[0]] = local_fixed.view(np.int64)           # bit pattern; torch has no uint64 collectives
    mine = torch.from_numpy(buf).to(device)
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine, group=group)
    out = np.zeros((n_events, width), dtype=np.uint64)
    for r, p in enumerate(parts):
        lo, hi = event_block(n_events, r, world)
        out[lo:hi] = p.cpu().numpy()[:hi - lo].view(np.uint64)
    return out


def max_over_ranks(value: float, group=None, device="cpu") -> float:
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t[0])


def sum_over_ranks(value: float, group=None, device="cpu") -> float:
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return float(t[0])
