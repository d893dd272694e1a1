"""Pins of the oracle's integer / indexing work (spec S2, S9) against an independent numpy restatement,
plus sort-mode invariance and per-event energy conservation on showers (pin 5). No GPU."""
import numpy as np
import pytest

import oracle as orc
from helpers import make_oracle
from paper_2503_17608_b200 import workloads as W

VACANT = 7
M_E = 0.51099895


def small_shower(sort_mode, n_slots=256, n_events=3, energy=200.0, seed=21, field=(1.0, 0.0, 0.0)):
    w = W.config2(n_events=n_events, n_slots=n_slots, sort_mode=sort_mode, seed=seed, energy=energy, field_T=field)
    return w, make_oracle(w)


@pytest.mark.parametrize("sort_mode", [0, 1, 2])
def test_init_sort_push_vs_numpy_restatement(sort_mode):
    w, o = small_shower(sort_mode, n_slots=64, n_events=4, energy=300.0)
    o.begin(w.primaries, w.n_events)
    n_iter = 0
    while n_iter < 400:
        before = o.state(); init_before = o.initializers()
        o.phase_init()
        after = o.state(); init_after = o.initializers()
        # --- S9: rank-r vacant slot (ascending) takes init[I-1-r]
        vac = np.flatnonzero(before["action"] == VACANT)
        n_take = min(len(vac), len(init_before))
        taken = vac[:n_take]
        src = init_before[::-1][:n_take]
        for f in ("pos", "dir", "energy", "event", "ptype", "vol", "surf"):
            assert np.array_equal(after[f][taken], src[f])
        assert np.all(after["nsteps"][taken] == 0)
        assert np.array_equal(after["action"][taken], np.where(src["ptype"] == 0, 3, 4))
        untouched = np.setdiff1d(np.arange(o.n_slots), taken)
        assert np.array_equal(after[untouched], before[untouched])
        assert len(init_after) == len(init_before) - n_take
        assert np.array_equal(init_after, init_before[:len(init_after)])
        # --- S2: stable counting sort = numpy stable argsort of the keys
        o.phase_reindex()
        idx, off = o.indices()
        act = after["action"]
        if sort_mode == 1:
            keys = act; nk = 8
        elif sort_mode == 2:
            keys = np.where(act == VACANT, 3, after["ptype"]); nk = 4
        else:
            keys = np.zeros_like(act); nk = 1
        assert np.array_equal(idx, np.argsort(keys, kind="stable").astype(np.uint32))
        cnt = np.bincount(keys, minlength=8)[:8]
        expect_off = np.concatenate([[0], np.cumsum(cnt[:nk])])
        assert np.array_equal(off[:nk + 1], expect_off)
        assert np.all(off[nk:] == off[nk])
        assert np.array_equal(o.counts()[-1], np.bincount(act, minlength=8))
        # --- S9 push: new initializers appended in ascending parent-slot order
        o.phase_rest()
        st = o.state(); init_new = o.initializers()[len(init_after):]
        if len(init_new):
            # parent of a secondary: the slot whose (frozen) position equals the secondary's birth position
            parent = []
            for s in init_new:
                m = np.flatnonzero(np.all(st["pos"] == s["pos"], axis=1) & (st["event"] == s["event"]))
                # a moved survivor no longer sits at the birth position; fall back to 'unknown'
                parent.append(int(m[0]) if len(m) else -1)
            known = [p for p in parent if p >= 0]
            assert known == sorted(known)
        n_iter += 1
        alive = (st["action"] != VACANT).sum()
        if alive == 0 and len(o.initializers()) == 0:
            break
    assert n_iter < 400
    T = o.tallies()
    assert np.abs(T.sum(1) - 300.0).max() < 1e-9 * 300.0


def test_tiny_hand_checkable_fill():
    """N = 8, 3 primaries: slots 0,1,2 take init[2], init[1], init[0]"""
    w = W.config1(n_events=3, n_slots=8)
    w.primaries["energy"] = [1.0, 2.0, 3.0]
    o = make_oracle(w)
    o.begin(w.primaries, 3)
    o.phase_init()
    st = o.state()
    assert list(st["energy"][:3]) == [3.0, 2.0, 1.0] and list(st["event"][:3]) == [2, 1, 0]
    assert np.all(st["action"][3:] == VACANT) and np.all(st["action"][:3] == 3)
    o.phase_reindex()
    idx, off = o.indices()
    assert list(idx) == [0, 1, 2, 3, 4, 5, 6, 7]
    assert list(off) == [0, 0, 0, 0, 3, 3, 3, 3, 8]


def test_partition_rule_hand_checkable():
    """S9-P (section 3.2): N = 8, all vacant, primaries 0..4 = gamma, e-, e-, gamma, e+. Pop order is
    init[4], init[3], ...: e+ -> lowest vacancy 0, gamma(3) -> highest vacancy 7, e-(2) -> 1, e-(1) -> 2, gamma(0) -> 6"""
    w = W.config2(n_events=5, n_slots=8, sort_mode=3, energy=100.0)
    w.primaries["ptype"] = [0, 1, 1, 0, 2]
    w.primaries["energy"] = [10.0, 11.0, 12.0, 13.0, 14.0]
    o = make_oracle(w)
    o.begin(w.primaries, 5)
    o.phase_init()
    st = o.state()
    assert list(st["energy"][[0, 1, 2, 6, 7]]) == [14.0, 12.0, 11.0, 10.0, 13.0]
    assert list(st["ptype"][[0, 1, 2, 6, 7]]) == [2, 1, 1, 0, 0]
    assert np.all(st["action"][3:6] == VACANT) and list(st["action"][[0, 1, 2, 6, 7]]) == [4, 4, 4, 3, 3]
    assert len(o.initializers()) == 0


def test_partition_rule_with_occupied_slots_and_starved_stack():
    """vacancies {1, 2, 4, 5, 7} of 8 slots (V = 5) and 7 initializers: the top 5 are popped; charged ones climb from
    the lowest vacancy, neutral ones descend from the highest, the other 2 stay on the stack in their order"""
    w = W.config2(n_events=10, n_slots=8, sort_mode=3, energy=100.0)
    w.primaries = w.primaries[:10].copy()
    w.primaries["ptype"] = [1, 1, 1, 0, 1, 0, 0, 1, 0, 1]        # first 3 fill slots 0.. in a plain run below
    w.primaries["energy"] = 20.0 + np.arange(10)
    o = make_oracle(w)
    o.begin(w.primaries, 10)
    o.phase_init()                                                # 8 slots <- top 8 (ids 9..2); stack keeps ids 0, 1
    st = o.state()
    # pop order ids 9(c) 8(g) 7(c) 6(g) 5(g) 4(c) 3(g) 2(c): charged -> 0,1,2,3 ; neutral -> 7,6,5,4
    assert list(st["energy"]) == [29.0, 27.0, 24.0, 22.0, 23.0, 25.0, 26.0, 28.0]
    assert [int(e) for e in o.initializers()["energy"]] == [20, 21]


def test_partition_mode_conserves_and_separates():
    """same physics in every mode: per-event energy is conserved; from an empty array the charged tracks of the first
    fill sit below every neutral one; a whole shower ends with the same number of histories' energy"""
    w, o = small_shower(3, n_slots=512, n_events=5, energy=500.0, seed=33)
    o.begin(w.primaries, w.n_events)
    for _ in range(6):
        o.step()
        st = o.state()
        ch = np.nonzero((st["action"] != VACANT) & (st["ptype"] != 0))[0]
        ne = np.nonzero((st["action"] != VACANT) & (st["ptype"] == 0))[0]
        if len(ch) and len(ne) and len(ch) + len(ne) < 200:      # far from full: no mixing yet
            assert ch.max() < ne.min()
    o.run()
    assert np.abs(o.tallies().sum(1) - 500.0).max() < 1e-9 * 500.0


def test_more_initializers_than_slots():
    w = W.config1(n_events=50, n_slots=16)
    o = make_oracle(w)
    o.begin(w.primaries, 50)
    o.phase_init()
    st = o.state()
    assert np.array_equal(st["event"], np.arange(49, 33, -1))
    assert len(o.initializers()) == 34
    o.phase_reindex(); o.phase_rest()
    o.run()
    assert np.abs(o.tallies().sum(1) - 1.0).max() < 1e-9


def test_sort_mode_invariance_bit_exact():
    """reindexing changes only the thread->slot map, not results (BASELINE.json config 3)"""
    res = []
    for mode in (0, 1, 2):
        w, o = small_shower(mode, n_slots=512, n_events=5, energy=500.0, seed=33)
        o.transport(w.primaries, w.n_events)
        res.append((o.tallies_fixed(), o.counts(), o.counters()))
    for r in res[1:]:
        assert np.array_equal(r[0], res[0][0])
        assert np.array_equal(r[1], res[0][1])
        assert r[2] == res[0][2]


@pytest.mark.parametrize("cfg", ["calo", "calo_field", "barrel"])
def test_energy_conservation_per_event(cfg):
    """pin 5: deposited + escaped = primary energy (+ 2 m_e per primary positron), per event, 1e-9 relative"""
    if cfg == "calo":
        w = W.config2(n_events=4, n_slots=1 << 12, energy=2000.0)
    elif cfg == "calo_field":
        w = W.config3(n_events=4, n_slots=1 << 12, energy=2000.0)
        w.primaries["ptype"][::2] = W.POSITRON
    else:
        w = W.config4(n_events=3, per_event=4, n_slots=1 << 12)
        w.primaries["energy"] *= 0.02
        # every volume with a material has a bin; vacuum volumes deposit nothing
    o = make_oracle(w)
    o.transport(w.primaries, w.n_events)
    T = o.tallies()
    expect = np.zeros(w.n_events)
    np.add.at(expect, w.primaries["event"], w.primaries["energy"] + np.where(w.primaries["ptype"] == 2, 2 * M_E, 0.0))
    assert np.abs(T.sum(1) - expect).max() < 1e-9 * expect.max()
    c = o.counters()
    cnt = o.counts()
    assert c["track_steps"] == int((w.n_slots - cnt[:, VACANT].astype(np.int64)).sum())
    assert np.all(cnt.sum(1) == w.n_slots)


def test_shower_shape_sanity():
    """parity unpinned externally: sanity only. 10 GeV in Pb/LAr: maximum near ln(E0/Ec) - 0.5 ~ 6.7 X0, contained"""
    w = W.config2(n_events=6, n_slots=1 << 14, energy=1e4)
    o = make_oracle(w)
    o.transport(w.primaries, w.n_events)
    T = o.tallies().sum(0)
    lay = T[:-1].reshape(50, 2).sum(1)
    x0_per_layer = 0.23 / 0.51372 + 0.57 / 14.1183
    tmax = (np.argmax(lay) + 0.5) * x0_per_layer
    assert 4.0 < tmax < 10.0
    assert T[:-1].sum() / T.sum() > 0.93
