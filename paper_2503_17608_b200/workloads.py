"""Seeded synthetic workloads (BASELINE.json configs 1-5) — input data only.

This module holds none of the method's arithmetic: it only builds the geometry / material /
physics descriptions and the primary particles, as plain numpy arrays and numbers, that are
handed identically to the CUDA path (paper_2503_17608_b200.binding) and to the CPU oracle
(oracle/oracle.py). It imports neither.

The paper measures on TestEM3 / CMS / ATLAS geometries with Geant4 physics data
(PAPER.md:89); none of that exists here, so these synthetic stand-ins (a 50-layer Pb/LAr
sampling calorimeter in 1 T for the TestEM3-like runs, a 3.8 T barrel for the CMS-like runs)
replace it — see DESIGN.md "input recipe".
"""
from dataclasses import dataclass, field

import numpy as np

PRIMARY_DTYPE = np.dtype([("event", "<u4"), ("ptype", "<i4"), ("energy", "<f8"), ("pos", "<f8", 3), ("dir", "<f8", 3)])
GAMMA, ELECTRON, POSITRON = 0, 1, 2
SORT_NONE, SORT_BY_ACTION, SORT_BY_PARTICLE, SORT_PARTITION, SORT_BY_ACTION_REUSE = 0, 1, 2, 3, 4

LEAD = (11.35, 82.0, 207.2)
LAR = (1.396, 18.0, 39.95)
SILICON = (2.33, 14.0, 28.09)
PBWO4 = (8.28, 73.0, 180.0)
BRASS = (8.53, 29.4, 63.5)


@dataclass
class Workload:
    name: str
    geometry: dict
    materials: list
    physics: dict
    n_slots: int
    sort_mode: int
    primaries: np.ndarray
    n_events: int
    notes: str = ""
    extra: dict = field(default_factory=dict)


def physics(seed, full=True, max_steps_per_track=2000, init_capacity=0):
    on = 1 if full else 0
    return dict(seed=int(seed), cut=1e-3, enable_pair=on, enable_brems=on, enable_msc=on, enable_eloss=on,
                enable_annihilation=on, electrons_local=0 if full else 1, max_substeps=10,
                max_steps_per_track=int(max_steps_per_track), init_capacity=int(init_capacity))


def beam(n_events, per_event, ptype, energy, pos=(0.0, 0.0, 0.0), direction=(0.0, 0.0, 1.0)):
    p = np.zeros(n_events * per_event, dtype=PRIMARY_DTYPE)
    p["event"] = np.repeat(np.arange(n_events, dtype=np.uint32), per_event)
    p["ptype"] = ptype
    p["energy"] = energy
    p["pos"] = pos
    p["dir"] = direction
    return p


def slab_geometry(bounds, vol_material, vol_bin, half, field_T=(0.0, 0.0, 0.0)):
    return dict(kind=0, bounds=np.asarray(bounds, np.float64), vol_material=np.asarray(vol_material, np.int32),
                vol_bin=np.asarray(vol_bin, np.int32), half_x=float(half), half_y=float(half), half_z=0.0,
                field=np.asarray(field_T, np.float64))


def calorimeter_geometry(field_T=(0.0, 0.0, 0.0), n_layers=50):
    """n_layers x (0.23 cm Pb + 0.57 cm LAr), 40 cm x 40 cm transverse (BASELINE.json config 2)."""
    bounds = []
    for i in range(n_layers):
        bounds += [0.8 * i, 0.8 * i + 0.23]
    bounds.append(0.8 * n_layers)
    mats = [0, 1] * n_layers
    bins = list(range(2 * n_layers))
    return slab_geometry(bounds, mats, bins, 20.0, field_T)


def barrel_geometry():
    """10 Si shells + PbWO4 + brass in 3.8 T along z (BASELINE.json config 4)."""
    bounds = [0.0]
    mats, bins = [], []
    b = 0
    for i in range(10):
        r = 3.0 + i * (107.0 / 9.0)
        bounds += [r, r + 0.03]
        mats += [-1, 0]; bins += [-1, b]; b += 1
    bounds += [129.0, 152.0]; mats += [-1, 1]; bins += [-1, b]; b += 1
    bounds += [180.0, 280.0]; mats += [-1, 2]; bins += [-1, b]; b += 1
    return dict(kind=1, bounds=np.asarray(bounds, np.float64), vol_material=np.asarray(mats, np.int32),
                vol_bin=np.asarray(bins, np.int32), half_x=0.0, half_y=0.0, half_z=300.0,
                field=np.asarray((0.0, 0.0, 3.8), np.float64))


def barrel_primaries(n_events, per_event, seed):
    """50/50 photons and electrons, log-uniform 1-100 GeV, |eta| < 2.5, uniform azimuth, from the origin.
    Draw order per primary: ln E, eta, phi from numpy Generator(PCG64(seed)); even index in event = photon."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = n_events * per_event
    draws = rng.random((n, 3))
    lnE = np.log(1e3) + draws[:, 0] * (np.log(1e5) - np.log(1e3))
    eta = -2.5 + 5.0 * draws[:, 1]
    phi = 2.0 * np.pi * draws[:, 2]
    theta = 2.0 * np.arctan(np.exp(-eta))
    p = np.zeros(n, dtype=PRIMARY_DTYPE)
    p["event"] = np.repeat(np.arange(n_events, dtype=np.uint32), per_event)
    p["ptype"] = np.where((np.arange(n) % per_event) % 2 == 0, GAMMA, ELECTRON)
    p["energy"] = np.exp(lnE)
    d = np.stack([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)], axis=1)
    p["dir"] = d / np.linalg.norm(d, axis=1, keepdims=True)
    return p


# ---------------------------------------------------------------- the five configs
def config1(n_events=1000, n_slots=4096, sort_mode=SORT_BY_ACTION, seed=1, energy=1.0):
    geo = slab_geometry([0.0, 1.0], [0], [0], 50.0)
    return Workload("photon_slab", geo, [LEAD], physics(seed, full=False), n_slots, sort_mode,
                    beam(n_events, 1, GAMMA, energy), n_events, "1 MeV photons into 1 cm Pb; KN + PE, electrons local")


def config2(n_events=1000, n_slots=1 << 20, sort_mode=SORT_BY_ACTION, seed=2, energy=1e4, field_T=(0.0, 0.0, 0.0), name="calorimeter"):
    geo = calorimeter_geometry(field_T)
    return Workload(name, geo, [LEAD, LAR], physics(seed), n_slots, sort_mode,
                    beam(n_events, 1, ELECTRON, energy), n_events, "10 GeV e- into 50 x (Pb 2.3 mm + LAr 5.7 mm)")


def config3(n_events=1000, n_slots=1 << 20, sort_mode=SORT_BY_ACTION, seed=3, energy=1e4):
    return config2(n_events, n_slots, sort_mode, seed, energy, field_T=(1.0, 0.0, 0.0), name="calorimeter_1T")


def config4(n_events=100, per_event=50, n_slots=1 << 22, sort_mode=SORT_BY_ACTION, seed=4):
    return Workload("barrel_3.8T", barrel_geometry(), [SILICON, PBWO4, BRASS], physics(seed), n_slots, sort_mode,
                    barrel_primaries(n_events, per_event, seed), n_events, "CMS-like barrel, mixed gamma/e- 1-100 GeV")


def config5(n_slots=1 << 20, sort_mode=SORT_BY_ACTION, n_events=2000, seed=5, energy=1e4):
    w = config3(n_events, n_slots, sort_mode, seed, energy)
    w.name = "sweep_calorimeter_1T"
    return w
