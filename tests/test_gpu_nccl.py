"""The multi-GPU code path of bench.py (events sharded over ranks, one final exchange of the integer
tallies) executed on a GPU with the NCCL backend: world_size 1 is all a one-GPU box allows, but it runs the same calls —
process-group initialisation on the device, all_reduce MAX / SUM, all_gather of the tally rows from device memory — that
`bench.py --gpus N` makes; the 2-rank logic (ragged blocks, merge order) is covered on gloo in tests/test_multi_rank.py."""
import os
import socket

import numpy as np
import pytest

from paper_2503_17608_b200 import workloads as W

pytestmark = pytest.mark.gpu


def test_nccl_world1_merge_and_reductions():
    import torch
    import torch.distributed as dist
    from paper_2503_17608_b200 import binding, sharding
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
    try:
        w = W.config3(n_events=9, n_slots=1 << 12, energy=300.0)
        local, n_local, lo = sharding.shard_primaries(w.primaries, w.n_events, 0, 1)
        assert n_local == w.n_events and lo == 0
        ctx = binding.from_workload(w)
        ctx.transport(local, n_local)
        v = ctx.tallies_view()
        merged = sharding.merge_tallies(v["fixed"], w.n_events, device=dev)          # all_gather on the device
        assert merged.dtype == np.uint64 and np.array_equal(merged, v["fixed"])
        assert sharding.max_over_ranks(12.5, device=dev) == 12.5                     # all_reduce MAX
        assert sharding.sum_over_ranks(float(v["track_steps"]), device=dev) == float(v["track_steps"])   # all_reduce SUM
        dist.barrier()
        ctx.close()
    finally:
        dist.destroy_process_group()
