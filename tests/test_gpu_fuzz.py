"""Randomised parity: seeded random geometries (slabs and cylinders of 1-12 volumes with vacuum gaps and unscored volumes,
thicknesses 0.1 mm - 5 cm), fields (none, along an axis, oblique), physics switches, substep and looper caps, slot
counts from "exactly the primaries" to 5000, all five sort modes, and primaries of all three species from 2 keV to 2 GeV
started inside volumes, ON boundaries and along the axes — stepped in lockstep with the oracle (integer work bit-exact,
floats 1e-12, tallies per iteration; later divergence only by float-driven decision flips: test_gpu_parity.lockstep).
The fixed configs of BASELINE.json exercise one geometry each; this walks the corners of the spec (S5-S7) they miss."""
import numpy as np
import pytest

from paper_2503_17608_b200 import workloads as W
from test_gpu_parity import lockstep

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2503_17608_b200 import binding as b
    b.load_library()
    return b


MATS = [W.LEAD, W.LAR, W.SILICON, W.PBWO4, W.BRASS]
def random_workload(rng):
    """input data only: none of the method's arithmetic"""
    kind = int(rng.integers(0, 2))
    n_vol = int(rng.integers(1, 13))
    n_mats = int(rng.integers(1, 4))
    mats = [MATS[i] for i in rng.choice(len(MATS), n_mats, replace=False)]
    th = np.exp(rng.uniform(np.log(0.01), np.log(5.0), n_vol))
    vm = rng.integers(-1, n_mats, n_vol).astype(np.int32)
    bins = np.where(rng.random(n_vol) < 0.2, -1, rng.integers(0, 4, n_vol)).astype(np.int32)
    fld = [(0, 0, 0), (1.0, 0, 0), (0, 0.5, 0), (0, 0, 3.8), (0.3, 0.4, 1.2)][int(rng.integers(0, 5))]
    if kind == 0:
        z0 = float(rng.uniform(-2, 2)); bounds = z0 + np.concatenate([[0.0], np.cumsum(th)])
        geo = W.slab_geometry(bounds, vm, bins, float(rng.uniform(0.5, 30.0)), fld)
    else:
        r0 = 0.0
        bounds = r0 + np.concatenate([[0.0], np.cumsum(th)])
        geo = dict(kind=1, bounds=np.asarray(bounds, np.float64), vol_material=vm, vol_bin=bins, half_x=0.0, half_y=0.0,
                   half_z=float(rng.uniform(0.5, 50.0)), field=np.asarray((0.0, 0.0, fld[2]) if rng.random() < 0.7 else fld, np.float64))
    n_ev = int(rng.integers(1, 6)); per = int(rng.integers(1, 9)); n = n_ev * per
    p = np.zeros(n, dtype=W.PRIMARY_DTYPE)
    p["event"] = np.repeat(np.arange(n_ev, dtype=np.uint32), per)
    p["ptype"] = rng.integers(0, 3, n)
    p["energy"] = np.exp(rng.uniform(np.log(2e-3), np.log(2e3), n))
    d = rng.normal(size=(n, 3)); d /= np.linalg.norm(d, axis=1, keepdims=True)
    axis = rng.random(n) < 0.3
    d[axis] = np.eye(3)[rng.integers(0, 3, axis.sum())] * rng.choice([-1.0, 1.0], axis.sum())[:, None]
    p["dir"] = d
    lo, hi = bounds[0], bounds[-1]
    if kind == 0:
        z = rng.uniform(lo, hi, n)
        onb = rng.random(n) < 0.3
        z[onb] = rng.choice(bounds, onb.sum())
        # a primary on the first / last plane must point inwards
        z = np.where((z <= lo) & (d[:, 2] <= 0), lo + 1e-3 * (hi - lo), z); z = np.where((z >= hi) & (d[:, 2] >= 0), hi - 1e-3 * (hi - lo), z)
        p["pos"] = np.stack([rng.uniform(-0.4, 0.4, n) * geo["half_x"], rng.uniform(-0.4, 0.4, n) * geo["half_y"], z], axis=1)
    else:
        r = rng.uniform(lo, hi * 0.999, n)
        phi = rng.uniform(0, 2 * np.pi, n)
        p["pos"] = np.stack([r * np.cos(phi), r * np.sin(phi), rng.uniform(-0.9, 0.9, n) * geo["half_z"]], axis=1)
    mode = int(rng.choice([0, 1, 2, 3, 4]))
    ph = W.physics(int(rng.integers(1, 1 << 30)), full=bool(rng.random() < 0.85), max_steps_per_track=int(rng.choice([50, 2000])))
    ph["max_substeps"] = int(rng.choice([1, 3, 10]))
    n_slots = int(rng.choice([n, 64, 777, 5000]))
    return W.Workload("fuzz", geo, mats, ph, n_slots, mode, p, n_ev, "fuzz")


@pytest.mark.parametrize("block", range(6))
def test_random_cases_in_lockstep(binding, block):
    for case in range(20):
        rng = np.random.default_rng(2503_17608 * 1000 + block * 20 + case)
        w = random_workload(rng)
        agreed = lockstep(binding, w, 40, must_match=1)
        assert agreed >= 1, (block, case)
