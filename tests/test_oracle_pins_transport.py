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
