"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (CUDA graph, batch 16, one launch
per action, default options): lockstep with the oracle over the first iterations at 2^20 slots, properties that hold
at any size on the whole run (per-event conservation, counter identities, sort-mode invariance, reproducibility), and
the per-layer profile of the full-energy run against an oracle sample of the same workload (3 sigma)."""
import numpy as np
import pytest

from helpers import make_oracle
from paper_2503_17608_b200 import workloads as W
from test_gpu_parity import lockstep, three_sigma, expected_energy, run_gpu, VACANT

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2503_17608_b200 import binding as b
    b.load_library()
    return b


def whole_run_properties(view, counts, w):
    e = view["fixed"].astype(np.float64).sum(1) * 2.0 ** -36
    want = expected_energy(w)
    assert np.all(np.abs(e - want) <= 1e-9 * want)                             # S10: per-event conservation
    alive = w.n_slots - counts[:, VACANT].astype(np.int64)
    assert np.all(counts.astype(np.int64).sum(1) == w.n_slots)                 # every slot has exactly one action
    assert view["track_steps"] == int(alive.sum())                             # S11
    assert view["iterations"] == int((alive > 0).sum())
    assert alive[0] == min(len(w.primaries), w.n_slots) and alive[-1] > 0


@pytest.mark.parametrize("cfg", ["config2", "config3"])
def test_calorimeter_full_size(binding, cfg):
    make = W.config2 if cfg == "config2" else W.config3
    w = make()                                                                  # 1000 x 10 GeV, 2^20 slots, by action
    assert w.n_slots == 1 << 20 and w.n_events == 1000 and w.sort_mode == 1
    # (1) the first iterations in lockstep with the oracle at the full slot count: integer work ==, floats 1e-12
    assert lockstep(binding, w, 5, must_match=3) >= 3
    # (2) the whole run as bench.py times it
    ref_view, ref_counts = run_gpu(binding, w)
    whole_run_properties(ref_view, ref_counts, w)
    again, again_counts = run_gpu(binding, w)
    assert np.array_equal(again["fixed"], ref_view["fixed"]) and np.array_equal(again_counts, ref_counts)   # reproducible
    for mode in (0, 2):                                                         # BASELINE.json config 3: bit-exact across sort modes
        w.sort_mode = mode
        v, c = run_gpu(binding, w)
        assert np.array_equal(v["fixed"], ref_view["fixed"]) and np.array_equal(c, ref_counts), mode
        assert v["track_steps"] == ref_view["track_steps"] and v["secondaries"] == ref_view["secondaries"]
    # (3) per-layer profile vs an oracle sample of the same workload, independent histories (other seed)
    wo = make(n_events=60, n_slots=1 << 17, seed=w.physics["seed"] + 100)
    o = make_oracle(wo)
    o.transport(wo.primaries, wo.n_events)
    z = three_sigma(ref_view["fixed"].astype(np.float64) * 2.0 ** -36, o.tallies())
    assert z.max() < 4.0, z.max()
    assert (z > 3.0).mean() <= 0.02 + 1.0 / len(z)


def test_barrel_full_size(binding):
    w = W.config4()                                                             # 100 events x 50, 2^22 slots, 3.8 T
    assert w.n_slots == 1 << 22 and w.n_events == 100
    view, counts = run_gpu(binding, w)
    whole_run_properties(view, counts, w)
    w.sort_mode = 0
    v, c = run_gpu(binding, w)
    assert np.array_equal(v["fixed"], view["fixed"]) and np.array_equal(c, counts)


def test_partition_full_size(binding):
    w = W.config3(sort_mode=3)
    assert lockstep(binding, w, 5, must_match=3) >= 3
    view, counts = run_gpu(binding, w)
    whole_run_properties(view, counts, w)
    wo = W.config3(n_events=60, n_slots=1 << 17, seed=w.physics["seed"] + 100, sort_mode=3)
    o = make_oracle(wo)
    o.transport(wo.primaries, wo.n_events)
    z = three_sigma(view["fixed"].astype(np.float64) * 2.0 ** -36, o.tallies())
    assert z.max() < 4.0 and (z > 3.0).mean() <= 0.02 + 1.0 / len(z)


def test_more_than_2048_tiles(binding):
    """above 2^22 slots the bookkeeping uses up to 4096 tiles (16 tile counters per thread in the block prefix, four
    warps of group rows): a ragged slot count there, in lockstep with the oracle and bit-identical across sort modes"""
    n_slots = (1 << 22) + 12345
    w = W.config3(n_events=60, n_slots=n_slots, energy=3000.0, seed=9)
    w.physics["init_capacity"] = 1 << 22
    assert lockstep(binding, w, 4, must_match=3) >= 3
    ref, ref_counts = run_gpu(binding, w)
    whole_run_properties(ref, ref_counts, w)
    for mode in (0, 2):
        w.sort_mode = mode
        v, c = run_gpu(binding, w)
        assert np.array_equal(v["fixed"], ref["fixed"]) and np.array_equal(c, ref_counts), mode


def test_maximum_slot_counts(binding):
    """n_slots up to the maximum cel_create accepts (2^28: 8192 bookkeeping tiles of 32 sub-tiles each, 57 GB of workspace):
    while the array never fills, tallies, counts and counters do not depend on the slot count (S9: ascending fill; S3:
    histories keyed by slot and iteration), so the runs at 2^26 and 2^28 slots must equal the run at 2^16 bit for bit —
    in every sort mode (the tiles of more than 4 sub-tiles re-read their key bytes for the scatter)"""
    def run(n_slots, mode):
        w = W.config3(n_events=20, n_slots=n_slots, energy=2000.0, seed=11, sort_mode=mode)
        w.physics["init_capacity"] = 1 << 22
        v, c = run_gpu(binding, w)
        return w, v, c
    refs = {}
    for mode in (1, 2, 4, 0):
        w, v, c = run(1 << 16, mode)
        whole_run_properties(v, c, w)
        assert c[:, :7].sum(1).max() < (1 << 16) // 4            # the premise, with room to spare
        refs[mode] = (v, c)
    for n_slots, modes in (((1 << 26) + 999, (1, 2, 4, 0)), (1 << 28, (1,))):
        for mode in modes:
            w, v, c = run(n_slots, mode)
            ref, cref = refs[mode]
            assert np.array_equal(v["fixed"], ref["fixed"]), (n_slots, mode)
            assert np.array_equal(c[:, :7], cref[:, :7]) and v["track_steps"] == ref["track_steps"] and v["secondaries"] == ref["secondaries"], (n_slots, mode)
            whole_run_properties(v, c, w)
