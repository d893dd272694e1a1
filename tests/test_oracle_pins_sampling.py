"""Pins of the oracle's samplers, geometry and helix against analytic distributions, brute force
and closed forms (spec S5-S8; BASELINE.json north_star pins 2 and 4). No GPU."""
import math

import numpy as np
import pytest
from scipy import integrate, stats

import oracle as orc
from helpers import golden_values, rel_close
from paper_2503_17608_b200 import workloads as W

G = golden_values()
M_E = 0.51099895
KAPPA = 2.99792458


# ---------------------------------------------------------------- Klein-Nishina sampler (pin 2)
def kn_pdf_eps(E, eps):
    k = E / M_E
    t = (1 - eps) / (k * eps)
    sin2 = t * (2 - t)
    return (1 / eps + eps) * (1 - eps * sin2 / (1 + eps * eps))


@pytest.mark.parametrize("E,tag", [(0.1, "0.1MeV"), (1.0, "1MeV"), (10.0, "10MeV")])
def test_kn_sampler_chi_square_and_moments(E, tag):
    n = 200000
    k = E / M_E
    e0 = 1 / (1 + 2 * k)
    eps = np.empty(n); cost = np.empty(n); trials = np.empty(n)
    for i in range(n):
        e, tt, s2, tr = orc.sample_kn(E, 77, i, 5)
        eps[i] = e; cost[i] = 1 - tt; trials[i] = tr
        if i < 2000:  # Compton kinematics identity E' = E / (1 + k (1 - cos theta)), and sin2 consistent
            assert abs(e - 1 / (1 + k * tt)) < 1e-13
            assert abs(s2 - (1 - (1 - tt) ** 2)) < 1e-13
    assert eps.min() >= e0 * (1 - 1e-12) and eps.max() <= 1.0
    norm, _ = integrate.quad(lambda x: kn_pdf_eps(E, x), e0, 1, epsrel=1e-12)
    edges = np.linspace(e0, 1, 51)
    expect = np.array([integrate.quad(lambda x: kn_pdf_eps(E, x), a, b, epsrel=1e-10)[0] for a, b in zip(edges[:-1], edges[1:])]) / norm * n
    obs, _ = np.histogram(eps, bins=edges)
    assert stats.chisquare(obs, expect * obs.sum() / expect.sum()).pvalue > 1e-3
    m_eps = integrate.quad(lambda x: x * kn_pdf_eps(E, x), e0, 1, epsrel=1e-12)[0] / norm
    m_cos = integrate.quad(lambda x: (1 - (1 - x) / (k * x)) * kn_pdf_eps(E, x), e0, 1, epsrel=1e-12)[0] / norm
    assert abs(m_eps - G[f"KN_mean_eps_{tag}"][0]) < 1e-7   # quadrature vs survey value
    assert abs(m_cos - G[f"KN_mean_cos_{tag}"][0]) < 1e-7
    assert abs(eps.mean() - m_eps) < 4 * eps.std() / math.sqrt(n)
    assert abs(cost.mean() - m_cos) < 4 * cost.std() / math.sqrt(n)
    # acceptance: 0.80 at 1 MeV, 0.99 at 100 MeV
    if E == 1.0:
        assert abs(1 / (1 + trials.mean()) - 0.80) < 0.02


def test_rotate_properties():
    rng = np.random.default_rng(3)
    for _ in range(500):
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        th = rng.uniform(0, math.pi); ph = rng.uniform(0, 2 * math.pi)
        out = orc.rotate(d, math.cos(th), math.sin(th), ph)
        assert abs(np.linalg.norm(out) - 1) < 1e-14
        assert abs(np.dot(out, d) - math.cos(th)) < 1e-13          # polar angle about d
    # azimuth convention: for d = +z the result is (sin th cos ph, sin th sin ph, cos th); for -z the z flips
    out = orc.rotate([0, 0, 1.0], math.cos(0.3), math.sin(0.3), 1.1)
    assert np.allclose(out, [math.sin(0.3) * math.cos(1.1), math.sin(0.3) * math.sin(1.1), math.cos(0.3)], atol=1e-15)
    out = orc.rotate([0, 0, -1.0], math.cos(0.3), math.sin(0.3), 1.1)
    assert np.allclose(out, [math.sin(0.3) * math.cos(1.1), math.sin(0.3) * math.sin(1.1), -math.cos(0.3)], atol=1e-15)
    # uniform phi gives directions uniform on the cone: mean of the transverse part vanishes
    d = np.array([0.6, 0.0, 0.8])
    acc = np.zeros(3)
    for ph in np.linspace(0, 2 * math.pi, 360, endpoint=False):
        acc += orc.rotate(d, math.cos(0.5), math.sin(0.5), ph)
    assert np.allclose(acc / 360, d * math.cos(0.5), atol=1e-12)


# ---------------------------------------------------------------- geometry vs brute-force ray marching
def _inside_slab(g, vol, p):
    return g["bounds"][vol] <= p[2] <= g["bounds"][vol + 1] and abs(p[0]) <= g["half_x"] and abs(p[1]) <= g["half_y"]


def _inside_cyl(g, vol, p):
    r = math.hypot(p[0], p[1])
    return g["bounds"][vol] <= r < g["bounds"][vol + 1] and abs(p[2]) <= g["half_z"]


def _march(inside, pos, d, smax):
    """first s where the ray leaves the volume: coarse march then bisection"""
    n = 4000
    prev = 0.0
    for i in range(1, n + 1):
        s = smax * i / n
        if not inside(pos + s * d):
            lo, hi = prev, s
            for _ in range(80):
                mid = 0.5 * (lo + hi)
                if inside(pos + mid * d):
                    lo = mid
                else:
                    hi = mid
            return 0.5 * (lo + hi)
        prev = s
    return None


def test_slab_distance_vs_ray_march():
    w = W.config2(n_events=1, n_slots=8)
    g = w.geometry
    o = orc.Oracle(g, w.materials, w.physics, 8, 1)
    rng = np.random.default_rng(5)
    for _ in range(300):
        vol = int(rng.integers(0, 100))
        z = rng.uniform(g["bounds"][vol], g["bounds"][vol + 1])
        pos = np.array([rng.uniform(-20, 20), rng.uniform(-20, 20), z])
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        s, which = o.distance(pos, d, vol, -1)
        ref = _march(lambda p: _inside_slab(g, vol, p), pos, d, 60.0)
        assert ref is not None and abs(s - ref) < 1e-9 * max(1.0, ref)
    # degenerate directions
    s, which = o.distance([0, 0, 0.1], [1.0, 0, 0], 0, -1)
    assert s == 20.0 and which == 2
    s, which = o.distance([0, 0, 0.23], [0, 0, -1.0], 1, -1)   # sitting on the plane it points at: zero-length crossing
    assert s == 0.0 and which == 1


def test_cylinder_distance_vs_ray_march():
    w = W.config4(n_events=1, per_event=2, n_slots=8)
    g = w.geometry
    o = orc.Oracle(g, w.materials, w.physics, 8, 1)
    rng = np.random.default_rng(6)
    nvol = len(g["vol_material"])
    for _ in range(300):
        vol = int(rng.integers(0, nvol))
        r = rng.uniform(g["bounds"][vol], g["bounds"][vol + 1])
        a = rng.uniform(0, 2 * math.pi)
        pos = np.array([r * math.cos(a), r * math.sin(a), rng.uniform(-299, 299)])
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        s, which = o.distance(pos, d, vol, -1)
        ref = _march(lambda p: _inside_cyl(g, vol, p), pos, d, 900.0)
        assert ref is not None and abs(s - ref) < 1e-9 * max(1.0, ref), (vol, s, ref)
    # on-surface logic: sitting on the inner surface of volume 3, moving outward -> only the outer is hit
    rin, rout = g["bounds"][3], g["bounds"][4]
    s, which = o.distance([rin, 0, 0], [1.0, 0, 0], 3, 3)
    assert which == 5 and abs(s - (rout - rin)) < 1e-12
    s, which = o.distance([rin, 0, 0], [-1.0, 0, 0], 3, 3)       # moving inward: zero-length re-crossing
    assert which == 4 and s == 0.0
    s, which = o.distance([rout, 0, 0], [1.0, 0, 0], 3, 4)       # on the outer, moving out
    assert which == 5 and s == 0.0
    s, which = o.distance([rout, 0, 0], [-1.0, 0, 0], 3, 4)      # on the outer, moving in: hits the inner first
    assert which == 4 and abs(s - (rout - rin)) < 1e-12
    # tangent-ish chord across volume 0 from its outer surface
    d = np.array([-math.cos(0.2), math.sin(0.2), 0.0])
    s, which = o.distance([g["bounds"][1], 0, 0], d, 0, 1)
    assert which == 5 and abs(s - 2 * g["bounds"][1] * math.cos(0.2)) < 1e-12
    # along the axis: only the end planes
    s, which = o.distance([1.0, 1.0, 10.0], [0, 0, 1.0], 0, -1)
    assert which == 1 and s == 290.0
    assert o.locate([0, 0, 0], [1.0, 0, 0]) == 0


# ---------------------------------------------------------------- helix (pin 4)
@pytest.mark.parametrize("T,B,key", [(1e4, 1.0, "helix_R_10GeV_1T_cm"), (1e4, 3.8, "helix_R_10GeV_3.8T_cm"), (1.0, 1.0, "helix_R_1MeV_1T_cm")])
def test_helix_radius_and_circle(T, B, key):
    p = math.sqrt(T * (T + 2 * M_E))
    R = p / (KAPPA * B)
    assert rel_close(R, *G[key])
    omega = -KAPPA * B / p              # electron
    bh = np.array([1.0, 0, 0])
    pos0 = np.array([0.3, -0.2, 0.1]); d0 = np.array([0.0, 0.0, 1.0])
    pts = [helix_pt for helix_pt in (orc.helix_point(pos0, d0, bh, omega, h)[0] for h in (0.0, 0.7 * R, 1.9 * R))]
    # circumradius of three points of the trajectory (generic geometry, independent of the helix formula)
    a = np.linalg.norm(pts[1] - pts[0]); b = np.linalg.norm(pts[2] - pts[1]); c = np.linalg.norm(pts[2] - pts[0])
    area = 0.5 * np.linalg.norm(np.cross(pts[1] - pts[0], pts[2] - pts[0]))
    assert rel_close(a * b * c / (4 * area), R, 1e-12)
    # sense of rotation: e- with B = +x, d = +z turns toward -y (F = q v x B)
    pe, de = orc.helix_point(pos0, d0, bh, omega, 0.01 * R)
    assert de[1] < 0 and pe[1] < pos0[1]
    pp, dp = orc.helix_point(pos0, d0, bh, -omega, 0.01 * R)   # positron
    assert dp[1] > 0
    # small-angle accuracy: 2 sin^2 form keeps full precision (10 GeV, h = 0.03 cm -> omega h ~ 1e-5)
    h = 0.03
    if abs(omega * h) < 1e-3:
        pe, de = orc.helix_point(np.zeros(3), d0, bh, omega, h)
        sag = h * h / (2 * R) * (1 - (omega * h) ** 2 / 12)     # series of R (1 - cos(h/R))
        assert abs(pe[1] + sag) < 1e-12 * sag                   # a naive 1 - cos would lose ~6 digits here


def test_helix_invariants_general_direction():
    rng = np.random.default_rng(8)
    for _ in range(200):
        bh = rng.normal(size=3); bh /= np.linalg.norm(bh)
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        pos = rng.normal(size=3)
        omega = rng.choice([-1, 1]) * 10 ** rng.uniform(-4, 1)
        h = 10 ** rng.uniform(-3, 1)
        p1, d1 = orc.helix_point(pos, d, bh, omega, h)
        assert abs(np.linalg.norm(d1) - 1) < 1e-13
        assert abs(np.dot(d1, bh) - np.dot(d, bh)) < 1e-13                # pitch conserved
        assert abs(np.dot(p1 - pos, bh) - h * np.dot(d, bh)) < 1e-12 * max(1, h)
        # composition: two half steps = one full step
        pm, dm = orc.helix_point(pos, d, bh, omega, 0.5 * h)
        p2, d2 = orc.helix_point(pm, dm, bh, omega, 0.5 * h)
        assert np.allclose(p2, p1, atol=1e-12 * max(1, h)) and np.allclose(d2, d1, atol=1e-12)
        # numerical derivative of position is the direction
        e = 1e-6 * min(h, 1 / abs(omega))
        pa, _ = orc.helix_point(pos, d, bh, omega, h + e); pb, _ = orc.helix_point(pos, d, bh, omega, h - e)
        assert np.allclose((pa - pb) / (2 * e), d1, atol=1e-6)
