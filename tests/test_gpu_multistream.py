"""Event-parallel multi-stream execution and the device-side timeline
(8(f)-4): K contexts on K streams driven by K host threads give, block by block, exactly what each
block gives when it is transported alone; the timeline is ordered like the iteration."""
import numpy as np
import pytest

from paper_2503_17608_b200 import sharding, workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2503_17608_b200 import binding as b
    b.load_library()
    return b


@pytest.mark.parametrize("k", [2, 3])
def test_blocks_equal_standalone_transports(binding, k):
    from paper_2503_17608_b200.multistream import MultiStream
    w = W.config3(n_events=12, n_slots=3 << 12, energy=300.0, seed=11)
    ms = MultiStream(w, k)
    ms.transport()
    fixed = ms.tallies_fixed()
    assert fixed.shape[0] == w.n_events
    total = ms.counters()
    steps = 0
    for r in range(k):
        prim, n_local, lo = sharding.shard_primaries(w.primaries, w.n_events, r, k)
        ctx = binding.from_workload(w, n_slots=w.n_slots // k)
        ctx.transport(prim, n_local)
        v = ctx.tallies_view()
        assert np.array_equal(v["fixed"], fixed[lo:lo + n_local]), r
        steps += v["track_steps"]
        ctx.close()
    assert steps == total["track_steps"]
    e = fixed.astype(np.float64).sum(1) * 2.0 ** -36
    assert np.all(np.abs(e - 300.0) <= 1e-9 * 300.0)     # energy conservation per event
    ms.close()


def test_timeline_is_ordered_and_does_not_change_results(binding):
    w = W.config2(n_events=8, n_slots=1 << 12, energy=200.0, seed=5)
    ctx = binding.from_workload(w)
    ctx.transport(w.primaries, w.n_events)
    ref = ctx.tallies_view()
    ref_fixed = ref["fixed"].copy()
    ctx.set_option("trace", 64)
    ctx.set_option("merge_discrete", 0)      # one launch per action, so that every action kernel has its own stamps
    ctx.transport(w.primaries, w.n_events)
    v = ctx.tallies_view()
    assert np.array_equal(v["fixed"], ref_fixed) and v["track_steps"] == ref["track_steps"]
    names, t = ctx.trace()
    assert names[0] == "fill_sort" and "push" in names and "discrete" in names and t.shape == (64, len(names), 2)
    n = min(64, int(v["iterations"]))
    t = t.astype(np.int64)
    ran = t[:n, :, 1] > 0
    i_fill, i_push = names.index("fill_sort"), names.index("push")
    assert ran[:, i_fill].all() and ran[:, i_push].all()
    assert ran[:, names.index("charged")].all() and not ran[:, names.index("discrete")].any()   # launch per action
    assert np.all(t[:n, :, 1][ran] >= t[:n, :, 0][ran])               # end >= start
    fill, push = t[:n, i_fill], t[:n, i_push]
    for j in range(len(names)):                                       # actions between P1 + P2 and P5
        if j in (i_fill, i_push):
            continue
        r = ran[:, j]
        assert np.all(t[:n, j, 0][r] >= fill[:, 1][r]) and np.all(push[:, 0][r] >= t[:n, j, 1][r])
    assert np.all(fill[1:, 0] >= push[:-1, 1])                        # next iteration after the push
    # the merged launch of the three pure interactions stamps "discrete" instead of their three kernels
    ctx.set_option("merge_discrete", 1)
    ctx.transport(w.primaries, w.n_events)
    v2 = ctx.tallies_view()
    assert np.array_equal(v2["fixed"], ref_fixed)
    _, t2 = ctx.trace()
    assert (t2[:n, names.index("discrete"), 1] > 0).all() and not (t2[:n, names.index("photoelectric"), 1] > 0).any()
    ctx.close()
