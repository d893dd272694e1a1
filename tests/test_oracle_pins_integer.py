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


def test_results_do_not_depend_on_the_slot_count_while_the_array_never_fills():
    """an invariant of S9 + S3: vacancies are filled in ascending slot order and a history is keyed by (seed, slot,
    iteration), so as long as live tracks + initializers never exceed the slots (the stack is emptied by every fill) the
    slot assignment — and with it every tally, count and counter — is the same whatever n_slots is"""
    res = []
    for n_slots in (1024, 1500, 4096):
        w, o = small_shower(1, n_slots=n_slots, n_events=5, energy=300.0, seed=33)
        o.transport(w.primaries, w.n_events)
        c = o.counts()
        assert (c[:, :7].sum(1).max()) < 1024                   # the premise: the smallest array never fills
        res.append((o.tallies_fixed(), c[:, :7].copy(), o.counters()))
    for r in res[1:]:
        assert np.array_equal(r[0], res[0][0]) and np.array_equal(r[1], res[0][1]) and r[2] == res[0][2]
    # and it does depend on it once the array fills (the premise is not vacuous)
    w, o = small_shower(1, n_slots=64, n_events=5, energy=300.0, seed=33)
    o.transport(w.primaries, w.n_events)
    assert not np.array_equal(o.tallies_fixed(), res[0][0])


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


# ---------------------------------------------------------------- S9-R: parent-slot reuse (sort mode 4)
def _block(mat_index=0):
    return W.slab_geometry([-1e6, 1e6], [mat_index], [0], 1e6)


def test_reuse_rule_hand_worked_photoelectric_and_annihilation():
    """hand-worked S9-R cases. (a) a 20 keV photon in Pb is absorbed photoelectrically (Sigma_PE / Sigma_tot > 0.999):
    its electron (T = E, same direction) appears IN THE PHOTON'S SLOT at the end of the absorbing iteration, nothing is
    pushed. (b) a positron below the cut stops (S7.1), annihilates in the next iteration: photon (m_e, u) takes the
    slot, photon (m_e, -u) is the only push."""
    p = W.physics(41)
    n = 64
    o = orc.Oracle(_block(), [W.LEAD], p, n, 4)
    prim = W.beam(n, 1, W.GAMMA, 0.02)
    o.begin(prim, n)
    o.step()                                  # move: every photon picks PE (or, rarely, Compton) at its interaction point
    st1 = o.state().copy()
    pe = st1["action"] == 0
    assert pe.sum() >= n - 2
    o.step()                                  # PE applied: electron in place
    st2 = o.state()
    assert len(o.initializers()) == 0 and o.counters()["secondaries"] == 0
    assert np.all(st2["ptype"][pe] == 1) and np.all(st2["action"][pe] == 4) and np.all(st2["nsteps"][pe] == 0)
    assert np.array_equal(st2["energy"][pe], st1["energy"][pe]) and np.array_equal(st2["pos"][pe], st1["pos"][pe])
    assert np.array_equal(st2["dir"][pe], st1["dir"][pe]) and np.array_equal(st2["event"][pe], st1["event"][pe])
    assert np.array_equal(st2["vol"][pe], st1["vol"][pe]) and np.array_equal(st2["surf"][pe], st1["surf"][pe])
    assert o.tallies().sum() == 0.0           # nothing deposited yet: the electrons are tracked
    # the same run in mode 1: the electrons go through the stack and come back in LIFO order
    o1 = orc.Oracle(_block(), [W.LEAD], p, n, 1)
    o1.begin(prim, n); o1.step(); o1.step()
    assert len(o1.initializers()) == pe.sum() and np.all(o1.state()["action"][pe] == VACANT)
    # (b)
    o = orc.Oracle(_block(), [W.LEAD], p, 4, 4)
    o.begin(W.beam(1, 1, W.POSITRON, 5e-4), 1)
    o.step()
    assert o.state()[0]["action"] == 6
    o.step()
    st = o.state()[0]; ini = o.initializers()
    assert st["action"] == 3 and st["ptype"] == 0 and st["energy"] == M_E and st["nsteps"] == 0
    assert len(ini) == 1 and ini[0]["energy"] == M_E and np.array_equal(ini[0]["dir"], -st["dir"])
    assert np.array_equal(ini[0]["pos"], st["pos"]) and o.counters()["secondaries"] == 1
    o.step()                                  # the pushed photon fills slot 1 (the lowest vacancy) in P1 of the next iteration
    assert o.state()[1]["event"] == 0 and len(o.initializers()) == 0
    o.run()
    assert abs(o.tallies().sum() - (5e-4 + 2 * M_E)) < 1e-9


def test_reuse_rule_hand_worked_pair():
    """a 50 MeV photon converts: e- (first staged) takes the slot, e+ is pushed; energies add up to E - 2 m_e"""
    n = 200
    E = 50.0
    o = orc.Oracle(_block(), [W.LEAD], W.physics(42), n, 4)
    o.begin(W.beam(n, 1, W.GAMMA, E), n)
    o.step()
    st1 = o.state().copy()
    pair = np.flatnonzero(st1["action"] == 1)
    assert len(pair) > 0.9 * n
    o.step()
    st2 = o.state(); ini = o.initializers()
    pos_of = {tuple(st1["pos"][s]): s for s in pair}
    eplus = [i for i in ini if i["ptype"] == 2]
    assert len(eplus) == len(pair)
    for i in eplus:
        s = pos_of[tuple(i["pos"])]
        assert st2["ptype"][s] == 1 and st2["action"][s] == 4 and st2["nsteps"][s] == 0     # the e- is in the slot
        assert abs(st2["energy"][s] + i["energy"] + 2 * M_E - E) < 1e-13 * E
        assert np.array_equal(st2["dir"][s], st1["dir"][s]) and np.array_equal(st2["pos"][s], st1["pos"][s])
    # pushes are in ascending parent-slot order
    parents = [pos_of[tuple(i["pos"])] for i in eplus]
    assert parents == sorted(parents)


def test_reuse_rule_vs_mode1_restatement_on_showers():
    """S9-R restated against the oracle's own mode 1 on the same iteration: the two modes are driven in lockstep from
    the same state (same slots -> same PRNG streams) until the first reuse; in that iteration mode 1's pushed
    initializers, minus the first secondary of every parent slot that ended VACANT, are mode 4's pushes, and exactly
    those first secondaries sit in their parents' slots (as the tracks P1 would have made of them)."""
    checked = 0
    for seed in (51, 52, 53, 54):
        w1 = W.config2(n_events=6, n_slots=256, sort_mode=1, seed=seed, energy=300.0, field_T=(1.0, 0.0, 0.0))
        w4 = W.config2(n_events=6, n_slots=256, sort_mode=4, seed=seed, energy=300.0, field_T=(1.0, 0.0, 0.0))
        a, b = make_oracle(w1), make_oracle(w4)
        a.begin(w1.primaries, 6); b.begin(w4.primaries, 6)
        for k in range(200):
            a.phase_init(); b.phase_init()
            a.phase_reindex(); b.phase_reindex()
            pre = a.state().copy()
            assert np.array_equal(pre, b.state())
            ia0, ib0 = len(a.initializers()), len(b.initializers())
            a.phase_rest(); b.phase_rest()
            sa, sb = a.state(), b.state()
            new_a, new_b = a.initializers()[ia0:], b.initializers()[ib0:]
            # parent slot of each of mode 1's pushes: the slot that held that position before the iteration
            pos_of = {tuple(pre["pos"][s]): s for s in np.flatnonzero(pre["action"] != VACANT)}
            parent = np.array([pos_of[tuple(i["pos"])] for i in new_a], dtype=np.int64)
            assert np.all(np.diff(parent) >= 0)
            first_of_parent = np.ones(len(new_a), bool)
            first_of_parent[1:] = parent[1:] != parent[:-1]
            reused = first_of_parent & (sa["action"][parent] == VACANT) if len(new_a) else first_of_parent
            expect_push = new_a[~reused]
            assert np.array_equal(new_b, expect_push)
            for i, s in zip(new_a[reused], parent[reused]):
                t = sb[s]
                assert t["action"] == (3 if i["ptype"] == 0 else 4) and t["nsteps"] == 0 and t["ptype"] == i["ptype"]
                for f in ("pos", "dir", "energy", "event", "vol", "surf"):
                    assert np.array_equal(t[f], i[f])
            others = np.setdiff1d(np.arange(256), parent[reused]) if len(new_a) else np.arange(256)
            assert np.array_equal(sa[others], sb[others])
            if reused.any():
                checked += int(reused.sum())
                break                                   # histories separate here
    assert checked >= 4


def test_reuse_mode_conserves_energy_and_is_sort_consistent():
    """mode 4 on whole showers: per-event conservation (pin 5), the index array is the stable sort by action, and the
    number of pushes drops against mode 1 by about the number of slot-vacating interactions"""
    w = W.config2(n_events=5, n_slots=512, sort_mode=4, seed=33, energy=500.0, field_T=(1.0, 0.0, 0.0))
    o = make_oracle(w)
    o.begin(w.primaries, w.n_events)
    for _ in range(30):
        o.phase_init(); o.phase_reindex()
        idx, off = o.indices()
        act = o.state()["action"]
        assert np.array_equal(idx, np.argsort(act, kind="stable").astype(np.uint32))
        assert np.array_equal(off, np.concatenate([[0], np.cumsum(np.bincount(act, minlength=8))]))
        o.phase_rest()
    o.run()
    assert np.abs(o.tallies().sum(1) - 500.0).max() < 1e-9 * 500.0
    w1 = W.config2(n_events=5, n_slots=512, sort_mode=1, seed=33, energy=500.0, field_T=(1.0, 0.0, 0.0))
    o1 = make_oracle(w1); o1.transport(w1.primaries, w1.n_events)
    c4, c1 = o.counters(), o1.counters()
    assert c4["secondaries"] < 0.8 * c1["secondaries"]
    assert abs(c4["track_steps"] - c1["track_steps"]) < 0.1 * c1["track_steps"]


def test_openmp_threads_do_not_change_results():
    """the oracle's per-slot phases on several host threads (bench.py's all-cores cpu_baseline leg) give bit-identical
    tallies, counts and counters: slots are independent and the PRNG is counter-based"""
    import os
    w = W.config3(n_events=6, n_slots=1 << 12, energy=800.0, seed=77)
    res = []
    for n in (1, max(2, min(8, os.cpu_count() or 2))):
        o = make_oracle(w)
        o.set_threads(n)
        o.transport(w.primaries, w.n_events)
        res.append((o.tallies_fixed(), o.counts(), o.counters(), o.state()))
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1]) and res[0][2] == res[1][2]
    assert np.array_equal(res[0][3], res[1][3])
