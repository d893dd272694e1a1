"""Event sharding over ranks, world_size 2 on gloo, CPU only: each rank transports its block of
events with the CPU oracle standing in for the device path; the merged tallies must equal, per event, what each block
gives when transported alone, conserve energy, and the timing reductions must be max / sum over ranks."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, n_events, out_dir):
    for p in (ROOT, os.path.join(ROOT, "oracle"), os.path.join(ROOT, "tests")):
        if p not in sys.path:
            sys.path.insert(0, p)
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from helpers import make_oracle
    from paper_2503_17608_b200 import sharding, workloads as W
    w = W.config1(n_events=n_events, n_slots=512)
    w.primaries["energy"] = 0.5 + 0.01 * w.primaries["event"]       # events distinguishable
    local, n_local, lo = sharding.shard_primaries(w.primaries, w.n_events, rank, world)
    assert n_local == sharding.event_block(n_events, rank, world)[1] - lo
    assert local["event"].min() == 0 and local["event"].max() == n_local - 1
    o = make_oracle(w)
    o.transport(local, n_local)
    fixed = np.rint(o.tallies() * 2.0 ** 36).astype(np.uint64)
    merged = sharding.merge_tallies(fixed, n_events)
    tmax = sharding.max_over_ranks(10.0 + rank)
    tsum = sharding.sum_over_ranks(float(o.counters()["track_steps"]))
    np.save(os.path.join(out_dir, f"merged_{rank}.npy"), merged)
    np.save(os.path.join(out_dir, f"local_{rank}.npy"), fixed)
    np.save(os.path.join(out_dir, f"red_{rank}.npy"), np.array([tmax, tsum, float(o.counters()["track_steps"])]))
    dist.destroy_process_group()


def test_event_blocks_partition():
    from paper_2503_17608_b200 import sharding
    for n in (0, 1, 7, 1000):
        for world in (1, 2, 3, 8):
            blocks = [sharding.event_block(n, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == n
            assert all(blocks[i][1] == blocks[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in blocks]
            assert max(sizes) - min(sizes) <= 1


@pytest.mark.timeout(300)
def test_two_ranks_gloo_merge(tmp_path):
    from paper_2503_17608_b200 import sharding
    world, n_events = 2, 37                       # odd: ragged blocks
    mp.spawn(_worker, args=(world, _free_port(), n_events, str(tmp_path)), nprocs=world, join=True)
    merged = [np.load(tmp_path / f"merged_{r}.npy") for r in range(world)]
    assert np.array_equal(merged[0], merged[1])   # every rank holds the same global tally
    for r in range(world):
        lo, hi = sharding.event_block(n_events, r, world)
        assert np.array_equal(merged[0][lo:hi], np.load(tmp_path / f"local_{r}.npy"))
    # per-event energy conservation of the merged tally: deposited + escaped = primary energy
    e = merged[0].astype(np.float64).sum(1) * 2.0 ** -36
    assert np.abs(e - (0.5 + 0.01 * np.arange(n_events))).max() < 1e-9
    red = [np.load(tmp_path / f"red_{r}.npy") for r in range(world)]
    assert red[0][0] == red[1][0] == 11.0         # max over ranks of 10 + rank
    assert red[0][1] == red[1][1] == red[0][2] + red[1][2]
