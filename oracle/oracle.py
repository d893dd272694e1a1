"""ctypes front end of the CPU oracle (oracle/cel_oracle.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module. It imports nothing from
paper_2503_17608_b200 (the CUDA path) and the CUDA path imports nothing from here.
A workload is passed in as plain numpy arrays / numbers (see Oracle.__init__).
"""
import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build as _build  # noqa: E402  (oracle/build.py)

ACTIONS = ("PE", "PAIR", "COMPTON", "MOVE_G", "MOVE_C", "BREMS", "ANNIH", "VACANT")
TABLES = {"compton": 0, "pe": 1, "pair": 2, "brems": 3, "range": 4}
N_GRID = 577

TRACK_DTYPE = np.dtype([("pos", "<f8", 3), ("dir", "<f8", 3), ("energy", "<f8"), ("event", "<u4"),
                        ("nsteps", "<u4"), ("vol", "<i4"), ("surf", "<i4"), ("ptype", "<i4"), ("action", "<i4")])
PRIMARY_DTYPE = np.dtype([("event", "<u4"), ("ptype", "<i4"), ("energy", "<f8"), ("pos", "<f8", 3), ("dir", "<f8", 3)])
assert TRACK_DTYPE.itemsize == 80 and PRIMARY_DTYPE.itemsize == 64


class _Material(C.Structure):
    _fields_ = [("density", C.c_double), ("Z", C.c_double), ("A", C.c_double)]


class _Geometry(C.Structure):
    _fields_ = [("kind", C.c_int), ("n_vol", C.c_int), ("bounds", C.POINTER(C.c_double)),
                ("vol_material", C.POINTER(C.c_int)), ("vol_bin", C.POINTER(C.c_int)),
                ("half_x", C.c_double), ("half_y", C.c_double), ("half_z", C.c_double), ("field", C.c_double * 3)]


class _Physics(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("cut", C.c_double), ("enable_pair", C.c_int), ("enable_brems", C.c_int),
                ("enable_msc", C.c_int), ("enable_eloss", C.c_int), ("enable_annihilation", C.c_int),
                ("electrons_local", C.c_int), ("max_substeps", C.c_int), ("max_steps_per_track", C.c_uint32),
                ("init_capacity", C.c_uint64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Geometry), C.POINTER(_Material), C.c_int, C.POINTER(_Physics), C.c_uint64, C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_n_bins.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]
        L.orc_begin.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32]
        L.orc_step.argtypes = [C.c_void_p]
        L.orc_phase_init.argtypes = [C.c_void_p]
        L.orc_phase_reindex.argtypes = [C.c_void_p]
        L.orc_phase_rest.argtypes = [C.c_void_p]
        L.orc_run.restype = C.c_int64
        L.orc_run.argtypes = [C.c_void_p, C.c_uint64]
        for name in ("orc_read_state", "orc_read_counts", "orc_read_initializers", "orc_read_tallies", "orc_read_counters"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p]
        L.orc_read_indices.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_n_iterations_logged.restype = C.c_uint64
        L.orc_n_iterations_logged.argtypes = [C.c_void_p]
        L.orc_n_initializers.restype = C.c_uint64
        L.orc_n_initializers.argtypes = [C.c_void_p]
        L.orc_philox.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_uniform.restype = C.c_double
        L.orc_uniform.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32]
        L.orc_sigma_kn.restype = C.c_double
        L.orc_sigma_kn.argtypes = [C.c_double]
        L.orc_stopping_power.restype = C.c_double
        L.orc_stopping_power.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_inv_X0.restype = C.c_double
        L.orc_inv_X0.argtypes = [C.c_void_p, C.c_int]
        L.orc_table.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.orc_lookup.restype = C.c_double
        L.orc_lookup.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double]
        L.orc_range_inverse.restype = C.c_double
        L.orc_range_inverse.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_sample_kn.restype = C.c_double
        L.orc_sample_kn.argtypes = [C.c_double, C.c_uint64, C.c_uint32, C.c_uint32, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_uint32)]
        L.orc_rotate.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_void_p]
        L.orc_distance.restype = C.c_double
        L.orc_distance.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_int)]
        L.orc_helix_point.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_locate.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


# ---------------------------------------------------------------- stateless unit functions (pins)
def philox(counter, key):
    c = np.asarray(counter, dtype=np.uint32); k = np.asarray(key, dtype=np.uint32); out = np.zeros(4, np.uint32)
    lib().orc_philox(_p(c), _p(k), _p(out))
    return out


def uniform(seed, slot, k, phase, j):
    return lib().orc_uniform(seed, slot, k, phase, j)


def sigma_kn(E):
    return lib().orc_sigma_kn(E)


def sample_kn(E, seed, slot, k):
    """-> (eps, tt, sin2, accepted trial index)"""
    tt = C.c_double(); s2 = C.c_double(); tr = C.c_uint32()
    eps = lib().orc_sample_kn(E, seed, slot, k, C.byref(tt), C.byref(s2), C.byref(tr))
    return eps, tt.value, s2.value, tr.value


def rotate(d, ct, st, phi):
    d = np.asarray(d, dtype=np.float64); out = np.zeros(3)
    lib().orc_rotate(_p(d), ct, st, phi, _p(out))
    return out


def helix_point(pos, d, bh, omega, h):
    pos = np.asarray(pos, dtype=np.float64); d = np.asarray(d, dtype=np.float64); bh = np.asarray(bh, dtype=np.float64)
    po = np.zeros(3); do = np.zeros(3)
    lib().orc_helix_point(_p(pos), _p(d), _p(bh), omega, h, _p(po), _p(do))
    return po, do


class Oracle:
    """One oracle context. Arguments are plain data:

    geometry: dict(kind=0|1, bounds, vol_material, vol_bin, half_x, half_y, half_z, field)
    materials: sequence of (density_g_cm3, Z, A)
    physics: dict with the OrcPhysics field names
    """

    def __init__(self, geometry, materials, physics, n_slots, sort_mode):
        L = lib()
        self._bounds = np.ascontiguousarray(geometry["bounds"], dtype=np.float64)
        self._vm = np.ascontiguousarray(geometry["vol_material"], dtype=np.int32)
        self._vb = np.ascontiguousarray(geometry["vol_bin"], dtype=np.int32)
        g = _Geometry()
        g.kind = int(geometry["kind"]); g.n_vol = len(self._vm)
        g.bounds = self._bounds.ctypes.data_as(C.POINTER(C.c_double))
        g.vol_material = self._vm.ctypes.data_as(C.POINTER(C.c_int))
        g.vol_bin = self._vb.ctypes.data_as(C.POINTER(C.c_int))
        g.half_x = geometry["half_x"]; g.half_y = geometry["half_y"]; g.half_z = geometry["half_z"]
        for i in range(3):
            g.field[i] = float(geometry["field"][i])
        mats = (_Material * len(materials))(*[_Material(*map(float, m)) for m in materials])
        ph = _Physics()
        for name, _ in _Physics._fields_:
            setattr(ph, name, physics[name])
        self.n_slots = int(n_slots)
        self.h = L.orc_create(C.byref(g), mats, len(materials), C.byref(ph), self.n_slots, int(sort_mode))
        self.n_bins = L.orc_n_bins(self.h)
        self.n_events = 0

    def set_threads(self, n):
        """host threads of the per-slot phases (OpenMP); results are bit-identical for any n"""
        lib().orc_set_threads(self.h, int(n))

    def close(self):
        if self.h:
            lib().orc_destroy(self.h); self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- run control
    def begin(self, primaries, n_events):
        prim = np.ascontiguousarray(primaries, dtype=PRIMARY_DTYPE)
        self.n_events = int(n_events)
        rc = lib().orc_begin(self.h, _p(prim), len(prim), self.n_events)
        if rc != 0:
            raise RuntimeError(f"orc_begin failed: {rc}")

    def step(self):
        rc = lib().orc_step(self.h)
        if rc != 0:
            raise RuntimeError(f"orc_step failed: {rc}")

    def phase_init(self):
        lib().orc_phase_init(self.h)

    def phase_reindex(self):
        lib().orc_phase_reindex(self.h)

    def phase_rest(self):
        rc = lib().orc_phase_rest(self.h)
        if rc != 0:
            raise RuntimeError(f"orc_phase_rest failed: {rc}")

    def run(self, max_iter=1 << 40):
        n = lib().orc_run(self.h, max_iter)
        if n < 0:
            raise RuntimeError(f"orc_run failed: {n}")
        return n

    def transport(self, primaries, n_events):
        self.begin(primaries, n_events)
        return self.run()

    # ---- readers
    def state(self):
        out = np.zeros(self.n_slots, dtype=TRACK_DTYPE); lib().orc_read_state(self.h, _p(out)); return out

    def indices(self):
        idx = np.zeros(self.n_slots, np.uint32); off = np.zeros(9, np.uint32)
        lib().orc_read_indices(self.h, _p(idx), _p(off)); return idx, off

    def counts(self):
        n = lib().orc_n_iterations_logged(self.h); out = np.zeros((n, 8), np.uint32)
        if n:
            lib().orc_read_counts(self.h, _p(out))
        return out

    def initializers(self):
        n = lib().orc_n_initializers(self.h); out = np.zeros(n, dtype=TRACK_DTYPE)
        if n:
            lib().orc_read_initializers(self.h, _p(out))
        return out

    def tallies_fixed(self):
        out = np.zeros((self.n_events, self.n_bins + 1), np.uint64); lib().orc_read_tallies(self.h, _p(out)); return out

    def tallies(self):
        """MeV, [n_events][n_bins+1]; last column = escaped"""
        return self.tallies_fixed().astype(np.float64) * 2.0 ** -36

    def counters(self):
        out = np.zeros(4, np.uint64); lib().orc_read_counters(self.h, _p(out))
        return dict(track_steps=int(out[0]), iterations=int(out[1]), secondaries=int(out[2]), iter=int(out[3]))

    # ---- unit functions that need material / geometry data
    def table(self, mat, which):
        out = np.zeros(N_GRID); lib().orc_table(self.h, mat, TABLES[which], _p(out)); return out

    def lookup(self, mat, which, E):
        return lib().orc_lookup(self.h, mat, TABLES[which], E)

    def range_inverse(self, mat, r):
        return lib().orc_range_inverse(self.h, mat, r)

    def stopping_power(self, mat, T):
        return lib().orc_stopping_power(self.h, mat, T)

    def inv_X0(self, mat):
        return lib().orc_inv_X0(self.h, mat)

    def distance(self, pos, d, vol, surf):
        pos = np.asarray(pos, dtype=np.float64); d = np.asarray(d, dtype=np.float64); w = C.c_int()
        s = lib().orc_distance(self.h, _p(pos), _p(d), vol, surf, C.byref(w))
        return s, w.value

    def locate(self, pos, d):
        pos = np.asarray(pos, dtype=np.float64); d = np.asarray(d, dtype=np.float64)
        return lib().orc_locate(self.h, _p(pos), _p(d))
