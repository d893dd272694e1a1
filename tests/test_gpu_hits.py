"""Per-iteration hit transfer (section 3.4): the hit records the host receives —
through the stream-ordered path (pinned ring buffers, a flush kernel after every iteration, a consumer thread one batch
behind) and through the paper's synchronous "before" path — re-accumulate to exactly the device tally; the transport's
results do not change; K event-parallel contexts each deliver their own block's hits."""
import numpy as np
import pytest

from paper_2503_17608_b200 import sharding, workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2503_17608_b200 import binding as b
    b.load_library()
    return b


def run(binding, w, **opts):
    ctx = binding.from_workload(w)
    for k, v in opts.items():
        ctx.set_option(k, v)
    ctx.transport(w.primaries, w.n_events)
    view = ctx.tallies_view()
    hits = ctx.hits_view() if opts.get("hits") else None
    return ctx, view, hits


@pytest.mark.parametrize("mode", [1, 2])
@pytest.mark.parametrize("cfg", ["calo_1T", "barrel", "photon_slab"])
def test_host_accumulated_hits_equal_device_tally(binding, mode, cfg):
    if cfg == "calo_1T":
        w = W.config3(n_events=20, n_slots=1 << 14, energy=2000.0)
    elif cfg == "barrel":
        w = W.config4(n_events=2, per_event=6, n_slots=1 << 14)
    else:
        w = W.config1(n_events=3000, n_slots=4096)
    ref_ctx, ref, _ = run(binding, w)
    ref_ctx.close()
    ctx, view, hits = run(binding, w, hits=mode, hit_tally=1, batch=8)
    assert np.array_equal(view["fixed"], ref["fixed"]) and view["track_steps"] == ref["track_steps"]   # results unchanged
    assert hits["fixed"] is not None and np.array_equal(hits["fixed"], view["fixed"])                 # the test of the transfer
    assert hits["q_sum"] == int(view["fixed"].astype(object).sum())
    assert hits["n_hits"] > 0 and hits["bytes_d2h"] == 16 * hits["n_hits"]
    # a second transport on the same context starts from zero again
    ctx.transport(w.primaries, w.n_events)
    v2 = ctx.tallies_view(); h2 = ctx.hits_view()
    assert np.array_equal(h2["fixed"], v2["fixed"]) and h2["n_hits"] == hits["n_hits"]
    ctx.close()


def test_hit_callback_sees_every_record_once(binding):
    w = W.config3(n_events=10, n_slots=1 << 13, energy=1000.0)
    ctx = binding.from_workload(w)
    ctx.set_option("hits", 1); ctx.set_option("batch", 4)
    acc = np.zeros((w.n_events, ctx.n_bins + 1), np.uint64)
    calls = []

    def on_hits(h):
        np.add.at(acc, (h["event"], h["bin"]), h["q"])
        calls.append(len(h))

    ctx.set_hit_callback(on_hits)
    ctx.transport(w.primaries, w.n_events)
    view = ctx.tallies_view(); hv = ctx.hits_view()
    assert np.array_equal(acc, view["fixed"]) and sum(calls) == hv["n_hits"] and len(calls) > 3
    ctx.set_hit_callback(None)
    ctx.close()


def test_hit_overflow_is_a_sticky_error(binding):
    w = W.config3(n_events=10, n_slots=1 << 13, energy=1000.0)
    ctx = binding.from_workload(w)
    ctx.set_option("hits", 1); ctx.set_option("hit_capacity", 256)
    with pytest.raises(binding.CelError) as ei:
        ctx.transport(w.primaries, w.n_events)
        ctx.tallies_view()
    assert ei.value.code == -10
    ctx.close()


def test_event_parallel_contexts_deliver_their_own_hits(binding):
    from paper_2503_17608_b200.multistream import MultiStream
    w = W.config3(n_events=12, n_slots=3 << 12, energy=300.0, seed=11)
    for mode in (1, 2):
        ms = MultiStream(w, 3, options={"hits": mode, "hit_tally": 1, "batch": 4})
        ms.transport()
        fixed = ms.tallies_fixed()
        got = np.concatenate([c.hits_view()["fixed"] for c, _, n, _ in ms.parts if n], axis=0)
        assert np.array_equal(got, fixed)
        ms.close()
