"""Transport-level pins of the oracle (BASELINE.json north_star pins 1, 3, 4, 5 and the integer work):
attenuation exp(-mu x), transported CSDA path = R(T0), helix in vacuum, brems/pair/annihilation/Highland
distributions, per-event energy conservation, init/sort/push vs an independent numpy restatement,
sort-mode invariance. No GPU."""
import math

import numpy as np
import pytest
from scipy import stats

import oracle as orc
from helpers import golden_values, make_oracle, rel_close
from paper_2503_17608_b200 import workloads as W

G = golden_values()
M_E = 0.51099895
VACANT = 7


def big_block(material, field=(0, 0, 0), second=None):
    """one huge slab volume (optionally a second one behind a plane at z = second[0])"""
    if second is None:
        return W.slab_geometry([-1e6, 1e6], [0], [0], 1e6, field)
    return W.slab_geometry([0.0, second[0], 1e6], [0, second[1]], [0, 1], 1e6, field)


def phys(seed, **kw):
    p = W.physics(seed)
    p.update(kw)
    return p


def test_attenuation_and_first_interaction_split():
    """pin 1: uncollided fraction through 1 cm Pb = exp(-mu), mu = 1.5713220545 /cm"""
    n = 200000
    w = W.config1(n_events=n, n_slots=1 << 15)
    o = make_oracle(w)
    o.transport(w.primaries, n)
    T = o.tallies()
    assert np.abs(T.sum(1) - 1.0).max() < 1e-9                       # pin 5 on config 1
    unc = int((T[:, 1] == 1.0).sum())
    pexp = math.exp(-G["mu_Pb_1MeV"][0] * 1.0)
    assert abs(pexp - 0.2077703) < 1e-6
    assert abs(unc - n * pexp) < 3 * math.sqrt(n * pexp * (1 - pexp))
    # first-interaction split PE : Compton = 0.63641 : 0.36359, from iteration-1 counts
    o.begin(w.primaries[:30000], 30000)
    o.step(); o.step()
    c = o.counts()[1]
    npe, nco = int(c[0]), int(c[2])
    f = npe / (npe + nco)
    assert abs(f - 0.63641) < 4 * math.sqrt(0.636 * 0.364 / (npe + nco))


def test_photon_free_path_is_exponential():
    geo = big_block(0)
    n = 20000
    o = orc.Oracle(geo, [W.LEAD], phys(11, electrons_local=1, enable_pair=0), n, 0)
    o.begin(W.beam(n, 1, W.GAMMA, 1.0), n)
    o.step()
    z = o.state()["pos"][:, 2]
    mu = G["mu_Pb_1MeV"][0]
    assert abs(z.mean() - 1 / mu) < 4 / mu / math.sqrt(n)
    assert stats.kstest(z, "expon", args=(0, 1 / mu)).pvalue > 1e-3


def test_transported_csda_path_equals_range():
    """pin 3 (transport half): eloss-only electrons in an infinite medium stop after exactly R(T0)"""
    for mat, T0 in ((W.LEAD, 10.0), (W.LAR, 3.0), (W.LEAD, 0.05)):
        o = orc.Oracle(big_block(0), [mat], phys(12, enable_brems=0, enable_msc=0), 4, 1)
        o.begin(W.beam(1, 1, W.ELECTRON, T0), 1)
        n = o.run()
        st = o.state()[0]
        assert st["action"] == VACANT
        R = o.lookup(0, "range", T0)
        assert rel_close(st["pos"][2], R, 1e-9)
        assert abs(o.tallies()[0, 0] - T0) < 1e-9 * T0                # all energy deposited
        # step function: first step is max(0.2 R, 0.01)
        o.begin(W.beam(1, 1, W.ELECTRON, T0), 1); o.step()
        assert rel_close(o.state()[0]["pos"][2], max(0.2 * R, 0.01) if R > 0.01 else R, 1e-12)


def test_helix_transport_in_vacuum_stays_on_circle():
    """pin 4 (transport half): e- 10 GeV, B = 1 T along x, vacuum: all substep end points on the circle, cap 10"""
    geo = W.slab_geometry([-1e6, 1e6], [-1], [-1], 1e6, (1.0, 0.0, 0.0))
    o = orc.Oracle(geo, [W.LEAD], phys(13), 2, 1)
    T = 1e4
    p = math.sqrt(T * (T + 2 * M_E)); R = p / 2.99792458
    assert rel_close(R, *G["helix_R_10GeV_1T_cm"])
    o.begin(W.beam(1, 1, W.ELECTRON, T), 1)
    hmax = min(math.sqrt(8 * 1e-3 * R), 0.5 * R)
    assert hmax * hmax / (8 * R) <= 1e-3 * (1 + 1e-12)                # chord sagitta bound delta
    centre = np.array([0.0, -R, 0.0])                                 # e- turns toward -y
    for k in range(1, 6):
        o.step()
        st = o.state()[0]
        assert st["action"] == 4 and st["energy"] == T               # vacuum: no loss, still moving
        assert abs(np.linalg.norm(st["pos"] - centre) - R) < 1e-12 * R
        assert abs(st["pos"][0]) < 1e-12 and abs(st["dir"][0]) < 1e-15
        assert abs(np.linalg.norm(st["dir"]) - 1) < 1e-15
        # paused after exactly 10 substeps of h_max: arc length travelled = 10 k hmax
        ang = math.atan2(st["pos"][2], st["pos"][1] + R)
        assert abs(ang * R - 10 * k * hmax) < 1e-9 * R


def test_brems_distance_and_spectrum():
    """eloss off -> the interaction always wins; distance ~ Exp(mfp), ln k uniform on [ln kc, ln T]"""
    n = 20000
    T = 10.0
    o = orc.Oracle(big_block(0), [W.LEAD], phys(14, enable_eloss=0, enable_msc=0), n, 1)
    o.begin(W.beam(n, 1, W.ELECTRON, T), n)
    o.step()
    st = o.state()
    assert np.all(st["action"] == 5)
    mfp = G["brems_mfp_Pb_10MeV_cm"][0]
    assert abs(st["pos"][:, 2].mean() - mfp) < 4 * mfp / math.sqrt(n)
    assert stats.kstest(st["pos"][:, 2], "expon", args=(0, mfp)).pvalue > 1e-3
    o.step()
    ini = o.initializers()
    assert len(ini) == n and np.all(ini["ptype"] == 0)
    u = (np.log(ini["energy"]) - math.log(1e-3)) / (math.log(T) - math.log(1e-3))
    assert u.min() > 0 and u.max() < 1
    assert stats.kstest(u, "uniform").pvalue > 1e-3
    # photon is collinear, born at the parent's position; parent keeps T - k
    st2 = o.state()
    assert np.array_equal(ini["dir"], np.tile([0.0, 0, 1.0], (n, 1)))
    assert np.allclose(np.sort(ini["pos"][:, 2]), np.sort(st["pos"][:, 2]), rtol=0, atol=0)
    # mean radiated energy per interaction = (T - kc)/ln(T/kc)
    assert abs(ini["energy"].mean() - (T - 1e-3) / math.log(T / 1e-3)) < 4 * ini["energy"].std() / math.sqrt(n)


def test_pair_sharing_and_energy_balance():
    n = 20000
    E = 50.0
    o = orc.Oracle(big_block(0), [W.LEAD], phys(15), n, 1)
    o.begin(W.beam(n, 1, W.GAMMA, E), n)
    o.step(); o.step()
    c = o.counts()[1]
    assert c[1] > 0.9 * (c[0] + c[1] + c[2])                          # pair dominates at 50 MeV in Pb
    ini = o.initializers()
    el = ini[ini["ptype"] == 1]; po = ini[ini["ptype"] == 2]
    # staging order e-, e+ and one e+ per pair
    pairs = [(a, b) for a, b in zip(ini[:-1], ini[1:]) if a["ptype"] == 1 and b["ptype"] == 2 and np.array_equal(a["pos"], b["pos"])]
    assert len(po) == c[1]                                            # the e+ is always staged
    assert len(po) - 3 <= len(pairs) <= len(po)                       # an e- below the cut is deposited instead (P ~ 2e-5)
    tot = np.array([a["energy"] + b["energy"] + 2 * M_E for a, b in pairs])
    assert np.abs(tot - E).max() < 1e-13 * E
    frac = np.array([a["energy"] / (E - 2 * M_E) for a, b in pairs])
    assert stats.kstest(frac, "uniform").pvalue > 1e-3


def test_highland_width():
    """10 GeV e- through 0.03 cm Pb: plane-angle rms = theta0 = 2.9316e-4 rad"""
    n = 40000
    geo = big_block(0, second=(0.03, 1))
    o = orc.Oracle(geo, [W.LEAD, W.LAR], phys(16, enable_brems=0), n, 1)
    o.begin(W.beam(n, 1, W.ELECTRON, 1e4), n)
    o.step()
    st = o.state()
    assert np.all(st["vol"] == 1) and np.all(st["pos"][:, 2] == 0.03)
    thx = st["dir"][:, 0] / st["dir"][:, 2]; thy = st["dir"][:, 1] / st["dir"][:, 2]
    th0 = G["highland_theta0_10GeV_Pb_0.03cm"][0]
    for a in (thx, thy):
        assert abs(a.std() / th0 - 1) < 4 / math.sqrt(2 * n)
        assert abs(a.mean()) < 4 * th0 / math.sqrt(n)
    assert stats.kstest(thx / th0, "norm").pvalue > 1e-3


def test_annihilation_at_rest():
    n = 20000
    o = orc.Oracle(big_block(0), [W.LEAD], phys(17), n, 1)
    o.begin(W.beam(n, 1, W.POSITRON, 5e-4), n)                        # below the cut: stops at once (S7.1)
    o.step()
    assert np.all(o.state()["action"] == 6)
    o.step()
    ini = o.initializers()
    assert len(ini) == 2 * n and np.all(ini["ptype"] == 0) and np.all(ini["energy"] == M_E)
    a, b = ini[0::2], ini[1::2]
    assert np.array_equal(a["dir"], -b["dir"]) and np.array_equal(a["pos"], b["pos"])
    assert np.abs(np.linalg.norm(a["dir"], axis=1) - 1).max() < 1e-15
    assert stats.kstest(a["dir"][:, 2], "uniform", args=(-1, 2)).pvalue > 1e-3
    assert stats.kstest(np.arctan2(a["dir"][:, 1], a["dir"][:, 0]), "uniform", args=(-math.pi, 2 * math.pi)).pvalue > 1e-3
    # energy bookkeeping: T deposited, 2 m_e radiated
    o.run()
    T = o.tallies()
    assert np.abs(T.sum(1) - (5e-4 + 2 * M_E)).max() < 1e-9


def test_compton_triangle_closes():
    """electron direction = normalise(E d - E' d') and |E d - E' d'| = p_e (momentum conservation)"""
    n = 5000
    E = 2.0
    o = orc.Oracle(big_block(0), [W.LEAD], phys(18, enable_pair=0), n, 1)
    o.begin(W.beam(n, 1, W.GAMMA, E), n)
    o.step()
    was_compton = o.state()["action"] == 2
    o.step()
    st = o.state(); ini = o.initializers()
    el = ini[ini["ptype"] == 1]
    # photons that survived Compton and electrons above the cut, matched by event
    by_event = {int(e["event"]): e for e in el}
    checked = 0
    for s in np.flatnonzero(was_compton):
        t = st[s]
        if t["action"] == VACANT or int(t["event"]) not in by_event:
            continue
        e = by_event[int(t["event"])]
        if e["energy"] + t["energy"] < E * (1 - 1e-12):   # the electron of a PE event, not this Compton
            continue
        pe = math.sqrt(e["energy"] * (e["energy"] + 2 * M_E))
        # the photon moved after scattering, its direction is the scattered one
        resid = E * np.array([0, 0, 1.0]) - t["energy"] * t["dir"] - pe * e["dir"]
        assert np.abs(resid).max() < 1e-12 * E
        checked += 1
    assert checked > 500


def test_dip_rule_no_boundary_ping_pong():
    """S7.3 dip rule (reading A27): an electron on a Pb/LAr plane whose tangent points shallowly into the
    LAr while the helix curves back towards the Pb must not oscillate between the two volumes with zero-length steps.
    Case found in config 3 (event 0, seed 3): T = 45.7 keV, d_z = -0.0082, B = 1 T along x. Pinned by what the
    mathematics fixes: the track stops by energy loss within a few steps (CSDA range of 46 keV is < 0.01 cm), all of
    its energy is deposited, nothing goes to the escape bin through the looper cap, and every step moves the track."""
    geo = W.slab_geometry([0.0, 14.4, 14.63], [1, 0], [0, 1], 20.0, (1.0, 0.0, 0.0))
    p = W.beam(1, 1, W.ELECTRON, 0.04572788, pos=(-1.9362439, 3.2664487, 14.4))
    d = np.array([-0.65087321, 0.75914261, -0.0081586]); d /= np.linalg.norm(d)
    p["dir"] = d
    o = orc.Oracle(geo, [W.LEAD, W.LAR], phys(3, enable_brems=0), 4, 1)
    o.begin(p, 1)
    last = None; stuck = 0; n = 0
    while n < 200:
        o.step(); n += 1
        st = o.state()[0]
        if st["action"] == VACANT:
            break
        cur = tuple(st["pos"])
        stuck = stuck + 1 if cur == last else 0
        assert stuck <= 1, "more than one consecutive zero-length step"
        last = cur
    assert n < 40
    T = o.tallies()[0]
    assert T[-1] == 0.0 and abs(T.sum() - 0.04572788) < 1e-9 * 0.04572788


def test_no_track_reaches_looper_cap_in_the_calorimeter():
    """config 3 has no vacuum: with the dip rule no history is ended by the 2000-step looper cap, so the run length is
    set by the shower (a few hundred iterations), not by a stuck track"""
    w = W.config3(n_events=6, n_slots=1 << 13)
    o = make_oracle(w)
    o.transport(w.primaries, w.n_events)
    assert o.counters()["iterations"] < 400


# ---------------------------------------------------------------- round-2 pins: bin attribution, looper cap, cylinder crossings
def _range_tables(o, mat=0):
    u = math.log(1e-3) + np.arange(577) * (math.log(10.0) / 64.0)
    return u, o.table(mat, "range")


def _eloss_numpy(o, mat, T0, s):
    """T0 - Rinv(R(T0) - s) restated with numpy's piecewise-linear interpolation of the (already pinned) range table:
    R is linear in u = ln T between nodes (S4), Rinv is the inverse of that lerp"""
    u, R = _range_tables(o, mat)
    r0 = np.interp(math.log(T0), u, R)
    return T0 - math.exp(np.interp(r0 - s, R, u))


def test_score_bin_is_the_pre_step_volume():
    """S10: the deposit of a step goes to the bin of the volume occupied at the START of the iteration, also when the
    step ends in the next volume or outside. Two volumes with distinct bins (Pb bin 0 | LAr bin 1), eloss-only
    electrons (no brems, no MSC: the step is deterministic) started 10 um before a plane."""
    geo = W.slab_geometry([0.0, 1.0, 2.0], [0, 1], [0, 1], 50.0)
    Q = 2.0 ** -36
    T0 = 10.0
    eps = 1e-3
    # (1) crossing Pb -> LAr: the whole T0 - T1 of the crossing step lands in bin 0, nothing in bin 1 or escape
    o = orc.Oracle(geo, [W.LEAD, W.LAR], phys(31, enable_brems=0, enable_msc=0), 4, 1)
    o.begin(W.beam(1, 1, W.ELECTRON, T0, pos=(0.0, 0.0, 1.0 - eps)), 1)
    o.step()
    st = o.state()[0]
    assert st["vol"] == 1 and st["pos"][2] == 1.0 and st["action"] == 4        # it did cross, and is still moving
    s_b = 1.0 - (1.0 - eps)                                                     # the subtraction the step performs
    dep = _eloss_numpy(o, 0, T0, s_b)
    T = o.tallies()[0]
    assert abs(T[0] - dep) <= 1e-12 * T0 + Q and dep > 1e-3                     # a real deposit (~ 12 keV), in the Pb bin
    assert T[1] == 0.0 and T[2] == 0.0
    assert abs(st["energy"] - (T0 - dep)) <= 1e-12 * T0
    # (2) the NEXT step starts in LAr: its deposit goes to bin 1 and bin 0 stays what it was
    T1 = st["energy"]
    o.step()
    Tn = o.tallies()[0]
    r_lar = np.interp(math.log(T1), *_range_tables(o, 1))
    s2 = max(0.2 * r_lar, 0.01)
    assert s2 < 1.0                                                             # stays inside the LAr volume
    assert Tn[0] == T[0] and Tn[2] == 0.0
    assert abs(Tn[1] - _eloss_numpy(o, 1, T1, s2)) <= 1e-12 * T0 + Q
    # (3) escape step from LAr: deposit in bin 1 (pre-step), remainder T1 in the escape bin, nothing in bin 0
    o.begin(W.beam(1, 1, W.ELECTRON, T0, pos=(0.0, 0.0, 2.0 - eps)), 1)
    o.step()
    assert o.state()[0]["action"] == VACANT
    T = o.tallies()[0]
    dep = _eloss_numpy(o, 1, T0, 2.0 - (2.0 - eps))
    assert T[0] == 0.0 and abs(T[1] - dep) <= 1e-12 * T0 + Q and abs(T[2] - (T0 - dep)) <= 1e-12 * T0 + Q
    # (4) an interaction deposit (photoelectric with local electrons) goes to the bin of the volume the photon is in:
    # half of the photons start in the Pb, half in the LAr; per event the deposit sits in the bin of the absorption point
    n = 4000
    o = orc.Oracle(geo, [W.LEAD, W.LAR], phys(32, electrons_local=1, enable_pair=0), n, 0)
    prim = W.beam(n, 1, W.GAMMA, 0.05, pos=(0.0, 0.0, 0.5))                      # 50 keV: photoelectric dominates
    prim["pos"][1::2, 2] = 1.5
    o.begin(prim, n)
    seen = {0: 0, 1: 0}
    for _ in range(6):
        pre = o.state().copy()
        before = o.tallies_fixed().copy()
        o.step()
        d = o.tallies_fixed().astype(np.int64) - before.astype(np.int64)
        pe = np.flatnonzero(pre["action"] == 0)                                  # slots that apply PE in this iteration
        for s in pe:
            ev, vol = int(pre["event"][s]), int(pre["vol"][s])
            assert d[ev, vol] > 0 and d[ev, 1 - vol] == 0
            seen[vol] += 1
    assert seen[0] > 1000 and seen[1] > 1000


@pytest.mark.parametrize("ptype,rest", [(W.ELECTRON, 0.0), (W.POSITRON, 2 * M_E)])
def test_looper_cap_fate(ptype, rest):
    """S7.6: a charged track that has made max_steps_per_track steps is ended, its kinetic energy (+ 2 m_e for e+,
    reading A16) credited to the ESCAPE bin. Vacuum + 1 T: nothing else can end the track."""
    geo = W.slab_geometry([-1e6, 1e6], [-1], [0], 1e6, (1.0, 0.0, 0.0))
    T = 1e4
    o = orc.Oracle(geo, [W.LEAD], phys(33, max_steps_per_track=5), 2, 1)
    o.begin(W.beam(1, 1, ptype, T), 1)
    for k in range(1, 5):
        o.step()
        st = o.state()[0]
        assert st["action"] == 4 and st["nsteps"] == k and o.tallies().sum() == 0.0
    o.step()
    st = o.state()[0]
    assert st["action"] == VACANT
    Tl = o.tallies()[0]
    assert Tl[0] == 0.0 and abs(Tl[1] - (T + rest)) <= 1e-12 * (T + rest)
    o.step()                                                                    # nothing left: the run is over
    assert o.tallies()[0, 1] == Tl[1] and len(o.initializers()) == 0


def _walk_photon(o, max_steps=20):
    """step a single photon in an all-vacuum geometry; returns [(vol, surf, x, y), ...] until it is gone"""
    out = []
    for _ in range(max_steps):
        o.step()
        st = o.state()[0]
        if st["action"] == VACANT:
            out.append(("escaped", float(st["pos"][0]), float(st["pos"][1])))
            break
        out.append((int(st["vol"]), int(st["surf"]), float(st["pos"][0]), float(st["pos"][1])))
    return out


def test_cylinder_crossing_sequences():
    """S6 cylinder crossings: the (vol, surf) transitions a photon goes through in concentric vacuum shells
    r = 1, 2, 3, 4 cm are fixed by circle-line geometry; written out by hand below (surf = index of the radial
    boundary the track sits on; crossing outwards vol+1, inwards vol-1)."""
    geo = dict(kind=1, bounds=np.array([0.0, 1.0, 2.0, 3.0, 4.0]), vol_material=np.full(4, -1, np.int32),
               vol_bin=np.array([0, 1, 2, 3], np.int32), half_x=0.0, half_y=0.0, half_z=100.0, field=np.zeros(3))
    o = orc.Oracle(geo, [W.LEAD], phys(34), 1, 1)
    # radially outwards from the axis
    o.begin(W.beam(1, 1, W.GAMMA, 1.0, pos=(0, 0, 0), direction=(1, 0, 0)), 1)
    seq = _walk_photon(o)
    assert [s[:2] for s in seq[:-1]] == [(1, 1), (2, 2), (3, 3)] and seq[-1][0] == "escaped"
    assert np.allclose([s[2] for s in seq[:-1]] + [seq[-1][1]], [1.0, 2.0, 3.0, 4.0], rtol=0, atol=1e-12)
    assert o.tallies()[0, 4] == 1.0 and o.tallies()[0, :4].sum() == 0.0
    # radially inwards from r = 3.5, through the axis and out on the other side
    o.begin(W.beam(1, 1, W.GAMMA, 1.0, pos=(3.5, 0, 0), direction=(-1, 0, 0)), 1)
    seq = _walk_photon(o)
    assert [s[:2] for s in seq[:-1]] == [(2, 3), (1, 2), (0, 1), (1, 1), (2, 2), (3, 3)] and seq[-1][0] == "escaped"
    assert np.allclose([s[2] for s in seq[:-1]] + [seq[-1][1]], [3.0, 2.0, 1.0, -1.0, -2.0, -3.0, -4.0], rtol=0, atol=1e-12)
    # a chord with impact parameter 1.5 cm: reaches shell 1 (1 <= r < 2) but not the core; the line y = 1.5 meets the
    # circle of radius rho at x = +-sqrt(rho^2 - 2.25)
    o.begin(W.beam(1, 1, W.GAMMA, 1.0, pos=(-3.5, 1.5, 0), direction=(1, 0, 0)), 1)
    assert o.locate((-3.5, 1.5, 0.0), (1.0, 0.0, 0.0)) == 3
    seq = _walk_photon(o)
    assert [s[:2] for s in seq[:-1]] == [(2, 3), (1, 2), (2, 2), (3, 3)] and seq[-1][0] == "escaped"
    xs = [-math.sqrt(6.75), -math.sqrt(1.75), math.sqrt(1.75), math.sqrt(6.75), math.sqrt(13.75)]
    assert np.allclose([s[2] for s in seq[:-1]] + [seq[-1][1]], xs, rtol=0, atol=1e-12)
    assert all(abs(s[3] - 1.5) < 1e-15 for s in seq[:-1])
    # a chord with impact parameter 2.5 cm stays in shells 2 and 3
    o.begin(W.beam(1, 1, W.GAMMA, 1.0, pos=(-3.0, 2.5, 0), direction=(1, 0, 0)), 1)
    seq = _walk_photon(o)
    assert [s[:2] for s in seq[:-1]] == [(2, 3), (3, 3)] and seq[-1][0] == "escaped"
    assert np.allclose([s[2] for s in seq[:-1]] + [seq[-1][1]], [-math.sqrt(2.75), math.sqrt(2.75), math.sqrt(9.75)], rtol=0, atol=1e-12)
    # the end planes: a photon along z leaves through z = +half_z without any radial crossing
    o.begin(W.beam(1, 1, W.GAMMA, 1.0, pos=(1.5, 0, 0), direction=(0, 0, 1)), 1)
    seq = _walk_photon(o)
    assert len(seq) == 1 and seq[0][0] == "escaped" and o.state()[0]["pos"][2] == 100.0
