"""Thin ctypes binding of the celstep C ABI (include/cel.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libcelstep.so. There is no CPU fallback: if the
library is missing or no CUDA device is present, the calls raise. PyTorch is only used by callers for
device memory and streams (pass `tensor.data_ptr()` / `torch.cuda.current_stream().cuda_stream`).
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("CELSTEP_LIB") or os.path.join(HERE, "libcelstep.so")   # (CELSTEP_LIB: another build of the same ABI, for A/B timing)

PRIMARY_DTYPE = np.dtype([("event", "<u4"), ("ptype", "<i4"), ("energy", "<f8"), ("pos", "<f8", 3), ("dir", "<f8", 3)])
TRACK_DTYPE = np.dtype([("pos", "<f8", 3), ("dir", "<f8", 3), ("energy", "<f8"), ("event", "<u4"),
                        ("nsteps", "<u4"), ("vol", "<i4"), ("surf", "<i4"), ("ptype", "<i4"), ("action", "<i4")])
TABLES = {"compton": 0, "pe": 1, "pair": 2, "brems": 3, "range": 4}
EXPORTS = ["cel_create", "cel_set_stream", "cel_workspace_bytes", "cel_set_workspace", "cel_transport",
           "cel_transport_device", "cel_tallies", "cel_destroy", "cel_strerror", "cel_last_cuda_error", "cel_set_option",
           "cel_debug_begin", "cel_debug_step", "cel_debug_read_state", "cel_debug_read_indices",
           "cel_debug_n_initializers", "cel_debug_read_initializers", "cel_debug_n_counts", "cel_debug_read_counts",
           "cel_debug_table", "cel_debug_uniforms", "cel_kernel_count", "cel_kernel_name", "cel_kernel_times", "cel_trace", "cel_debug_math",
           "cel_set_hit_callback", "cel_hit_tallies", "cel_reindex_static", "cel_reindex_static_max_slots"]


class cel_material(C.Structure):
    _fields_ = [("density_g_cm3", C.c_double), ("Z", C.c_double), ("A", C.c_double)]


class cel_geometry(C.Structure):
    _fields_ = [("kind", C.c_int), ("n_vol", C.c_int), ("bounds", C.POINTER(C.c_double)),
                ("vol_material", C.POINTER(C.c_int)), ("vol_bin", C.POINTER(C.c_int)),
                ("half_x", C.c_double), ("half_y", C.c_double), ("half_z", C.c_double), ("field_T", C.c_double * 3)]


class cel_physics(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("cut_MeV", C.c_double), ("enable_pair", C.c_int), ("enable_brems", C.c_int),
                ("enable_msc", C.c_int), ("enable_eloss", C.c_int), ("enable_annihilation", C.c_int),
                ("electrons_local", C.c_int), ("max_substeps", C.c_int), ("max_steps_per_track", C.c_uint32),
                ("init_capacity", C.c_uint64)]


class cel_tally_view(C.Structure):
    _fields_ = [("n_events", C.c_uint32), ("n_bins", C.c_int32), ("fixed", C.POINTER(C.c_uint64)),
                ("track_steps", C.c_uint64), ("iterations", C.c_uint64), ("secondaries", C.c_uint64),
                ("seconds", C.c_double), ("kernel_launches", C.c_uint64)]


class cel_hit_view(C.Structure):
    _fields_ = [("n_hits", C.c_uint64), ("q_sum", C.c_uint64), ("bytes_d2h", C.c_uint64), ("n_events", C.c_uint32),
                ("n_bins", C.c_int32), ("fixed", C.POINTER(C.c_uint64))]


HIT_DTYPE = np.dtype([("event", "<u4"), ("bin", "<i4"), ("q", "<u8")])
HIT_CALLBACK = C.CFUNCTYPE(None, C.c_void_p, C.c_uint64, C.c_void_p)


class CelError(RuntimeError):
    def __init__(self, code, what, detail=""):
        super().__init__(f"{what}: {code} ({detail})")
        self.code = code


_lib = None


def load_library():
    """dlopen libcelstep.so and declare the signatures; raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(f"{LIB_PATH} is missing: run `python -m paper_2503_17608_b200.build` (there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    L.cel_create.argtypes = [C.POINTER(cel_geometry), C.POINTER(cel_material), C.c_int, C.POINTER(cel_physics), C.c_uint64, C.c_int, C.POINTER(vp)]
    L.cel_set_stream.argtypes = [vp, vp]
    L.cel_workspace_bytes.restype = C.c_uint64
    L.cel_workspace_bytes.argtypes = [C.c_uint64, C.c_uint64, C.c_int]
    L.cel_set_workspace.argtypes = [vp, vp, C.c_uint64]
    L.cel_transport.argtypes = [vp, vp, C.c_uint64, C.c_uint32]
    L.cel_transport_device.argtypes = [vp, vp, C.c_uint64, C.c_uint32]
    L.cel_tallies.argtypes = [vp, C.POINTER(cel_tally_view)]
    L.cel_destroy.argtypes = [vp]
    L.cel_destroy.restype = None
    L.cel_strerror.restype = C.c_char_p
    L.cel_strerror.argtypes = [C.c_int]
    L.cel_last_cuda_error.restype = C.c_char_p
    L.cel_last_cuda_error.argtypes = [vp]
    L.cel_set_option.argtypes = [vp, C.c_char_p, C.c_int64]
    L.cel_debug_begin.argtypes = [vp, vp, C.c_uint64, C.c_uint32]
    L.cel_debug_step.argtypes = [vp]
    L.cel_debug_read_state.argtypes = [vp, vp]
    L.cel_debug_read_indices.argtypes = [vp, vp, vp]
    L.cel_debug_n_initializers.argtypes = [vp, C.POINTER(C.c_uint64)]
    L.cel_debug_read_initializers.argtypes = [vp, vp]
    L.cel_debug_n_counts.argtypes = [vp, C.POINTER(C.c_uint64)]
    L.cel_debug_read_counts.argtypes = [vp, vp]
    L.cel_debug_table.argtypes = [vp, C.c_int, C.c_int, vp]
    L.cel_debug_uniforms.argtypes = [vp, vp, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, vp]
    L.cel_kernel_count.restype = C.c_int
    L.cel_kernel_name.restype = C.c_char_p
    L.cel_kernel_name.argtypes = [C.c_int]
    L.cel_kernel_times.argtypes = [vp, vp, vp]
    L.cel_trace.argtypes = [vp, vp, vp]
    L.cel_set_hit_callback.argtypes = [vp, HIT_CALLBACK, vp]
    L.cel_hit_tallies.argtypes = [vp, C.POINTER(cel_hit_view)]
    L.cel_reindex_static.argtypes = [vp, C.c_uint64, vp, vp, vp]
    L.cel_reindex_static_max_slots.restype = C.c_uint64
    L.cel_reindex_static_max_slots.argtypes = []
    _lib = L
    return L


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


class Context:
    """cel_ctx wrapper. geometry / materials / physics are the plain data of paper_2503_17608_b200.workloads."""

    def __init__(self, geometry, materials, physics, n_slots, sort_mode, stream=None, workspace=None, workspace_bytes=0):
        L = load_library()
        self._bounds = np.ascontiguousarray(geometry["bounds"], dtype=np.float64)
        self._vm = np.ascontiguousarray(geometry["vol_material"], dtype=np.int32)
        self._vb = np.ascontiguousarray(geometry["vol_bin"], dtype=np.int32)
        g = cel_geometry()
        g.kind = int(geometry["kind"]); g.n_vol = len(self._vm)
        g.bounds = self._bounds.ctypes.data_as(C.POINTER(C.c_double))
        g.vol_material = self._vm.ctypes.data_as(C.POINTER(C.c_int))
        g.vol_bin = self._vb.ctypes.data_as(C.POINTER(C.c_int))
        g.half_x = geometry["half_x"]; g.half_y = geometry["half_y"]; g.half_z = geometry["half_z"]
        for i in range(3):
            g.field_T[i] = float(geometry["field"][i])
        mats = (cel_material * len(materials))(*[cel_material(*map(float, m)) for m in materials])
        ph = cel_physics()
        ph.seed = physics["seed"]; ph.cut_MeV = physics["cut"]
        for k in ("enable_pair", "enable_brems", "enable_msc", "enable_eloss", "enable_annihilation", "electrons_local",
                  "max_substeps", "max_steps_per_track", "init_capacity"):
            setattr(ph, k, physics[k])
        self.n_slots = int(n_slots)
        self.sort_mode = int(sort_mode)
        h = C.c_void_p()
        self._check(L.cel_create(C.byref(g), mats, len(materials), C.byref(ph), self.n_slots, self.sort_mode, C.byref(h)), "cel_create", None)
        self.h = h
        self.n_events = 0
        self.n_bins = int(self._vb.max()) + 1 if len(self._vb) else 0
        if stream is not None:
            self.set_stream(stream)
        if workspace is not None:
            self.set_workspace(workspace, workspace_bytes)

    def _check(self, rc, what, h="self"):
        if rc != 0:
            L = load_library()
            detail = L.cel_strerror(rc).decode()
            hh = self.h if h == "self" else None
            if hh:
                detail += "; " + L.cel_last_cuda_error(hh).decode()
            raise CelError(rc, what, detail)

    def close(self):
        if getattr(self, "h", None):
            load_library().cel_destroy(self.h); self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the boundary calls, same names as include/cel.h
    def set_stream(self, cuda_stream: int):
        self._check(load_library().cel_set_stream(self.h, C.c_void_p(cuda_stream)), "cel_set_stream")

    def set_workspace(self, dptr: int, nbytes: int):
        self._check(load_library().cel_set_workspace(self.h, C.c_void_p(dptr), nbytes), "cel_set_workspace")

    def set_option(self, name: str, value: int):
        self._check(load_library().cel_set_option(self.h, name.encode(), int(value)), "cel_set_option")

    def transport(self, primaries, n_events):
        prim = np.ascontiguousarray(primaries, dtype=PRIMARY_DTYPE)
        self.n_events = int(n_events)
        self._check(load_library().cel_transport(self.h, _p(prim), len(prim), self.n_events), "cel_transport")

    def transport_device(self, d_primaries_ptr: int, n_primaries: int, n_events: int):
        self.n_events = int(n_events)
        self._check(load_library().cel_transport_device(self.h, C.c_void_p(d_primaries_ptr), int(n_primaries), self.n_events), "cel_transport_device")

    def tallies_view(self):
        v = cel_tally_view()
        self._check(load_library().cel_tallies(self.h, C.byref(v)), "cel_tallies")
        n = v.n_events * (v.n_bins + 1)
        fixed = np.ctypeslib.as_array(v.fixed, shape=(n,)).reshape(v.n_events, v.n_bins + 1).copy()
        return dict(fixed=fixed, track_steps=int(v.track_steps), iterations=int(v.iterations), secondaries=int(v.secondaries),
                    seconds=float(v.seconds), kernel_launches=int(v.kernel_launches), n_bins=int(v.n_bins))

    def tallies_fixed(self):
        return self.tallies_view()["fixed"]

    def tallies(self):
        """MeV, [n_events][n_bins+1]; last column = escaped energy"""
        return self.tallies_fixed().astype(np.float64) * 2.0 ** -36

    def kernel_times(self):
        """{kernel name: (device ms, launches)} of the last transport run with option profile=1"""
        L = load_library()
        n = L.cel_kernel_count()
        ms = np.zeros(n); cnt = np.zeros(n, np.uint64)
        self._check(L.cel_kernel_times(self.h, _p(ms), _p(cnt)), "cel_kernel_times")
        return {L.cel_kernel_name(i).decode(): (float(ms[i]), int(cnt[i])) for i in range(n)}

    def trace(self):
        """(kernel names, stamps[n_iters][n_kernels][2] uint64 ns) of the last transport run with option trace=n"""
        L = load_library()
        n = C.c_uint64(0)
        self._check(L.cel_trace(self.h, None, C.byref(n)), "cel_trace")
        out = np.zeros((n.value, L.cel_kernel_count(), 2), np.uint64)
        if n.value:
            self._check(L.cel_trace(self.h, _p(out), C.byref(n)), "cel_trace")
        return [L.cel_kernel_name(i).decode() for i in range(L.cel_kernel_count())], out

    def set_hit_callback(self, fn):
        """fn(hits: numpy structured array view (HIT_DTYPE), valid during the call) or None; called per batch of iterations"""
        if fn is None:
            self._hit_cb = HIT_CALLBACK(0)
        else:
            def tramp(ptr, n, _user):
                buf = (C.c_char * (int(n) * HIT_DTYPE.itemsize)).from_address(ptr)
                fn(np.frombuffer(buf, dtype=HIT_DTYPE))
            self._hit_cb = HIT_CALLBACK(tramp)
        self._check(load_library().cel_set_hit_callback(self.h, self._hit_cb, None), "cel_set_hit_callback")

    def hits_view(self):
        v = cel_hit_view()
        self._check(load_library().cel_hit_tallies(self.h, C.byref(v)), "cel_hit_tallies")
        fixed = None
        if v.fixed:
            n = v.n_events * (v.n_bins + 1)
            fixed = np.ctypeslib.as_array(v.fixed, shape=(n,)).reshape(v.n_events, v.n_bins + 1).copy()
        return dict(n_hits=int(v.n_hits), q_sum=int(v.q_sum), bytes_d2h=int(v.bytes_d2h), fixed=fixed)

    # ---- debug / parity surface
    def begin(self, primaries, n_events):
        prim = np.ascontiguousarray(primaries, dtype=PRIMARY_DTYPE)
        self.n_events = int(n_events)
        self._check(load_library().cel_debug_begin(self.h, _p(prim), len(prim), self.n_events), "cel_debug_begin")

    def step(self):
        self._check(load_library().cel_debug_step(self.h), "cel_debug_step")

    def state(self):
        out = np.zeros(self.n_slots, dtype=TRACK_DTYPE)
        self._check(load_library().cel_debug_read_state(self.h, _p(out)), "cel_debug_read_state")
        return out

    def indices(self):
        idx = np.zeros(self.n_slots, np.uint32); off = np.zeros(9, np.uint32)
        self._check(load_library().cel_debug_read_indices(self.h, _p(idx), _p(off)), "cel_debug_read_indices")
        return idx, off

    def initializers(self):
        n = C.c_uint64()
        self._check(load_library().cel_debug_n_initializers(self.h, C.byref(n)), "cel_debug_n_initializers")
        out = np.zeros(n.value, dtype=TRACK_DTYPE)
        if n.value:
            self._check(load_library().cel_debug_read_initializers(self.h, _p(out)), "cel_debug_read_initializers")
        return out

    def counts(self):
        n = C.c_uint64()
        self._check(load_library().cel_debug_n_counts(self.h, C.byref(n)), "cel_debug_n_counts")
        out = np.zeros((n.value, 8), np.uint32)
        if n.value:
            self._check(load_library().cel_debug_read_counts(self.h, _p(out)), "cel_debug_read_counts")
        return out

    def table(self, material, which):
        out = np.zeros(577)
        self._check(load_library().cel_debug_table(self.h, material, TABLES[which], _p(out)), "cel_debug_table")
        return out

    def uniforms(self, slots, k, phase, j):
        s = np.ascontiguousarray(slots, dtype=np.uint32); out = np.zeros(len(s))
        self._check(load_library().cel_debug_uniforms(self.h, _p(s), len(s), k, phase, j, _p(out)), "cel_debug_uniforms")
        return out

    def debug_math(self, which, x):
        """the path's small-angle sin (which=0) and 1 - cos (1) of the helix substep, evaluated on the device"""
        a = np.ascontiguousarray(x, dtype=np.float64); out = np.zeros(len(a))
        self._check(load_library().cel_debug_math(self.h, int(which), _p(a), len(a), _p(out)), "cel_debug_math")
        return out


def reindex_static_max_slots():
    return int(load_library().cel_reindex_static_max_slots())


def reindex_static(d_keys_ptr: int, n_slots: int, d_indices_ptr: int, d_offsets_ptr: int, stream: int = 0):
    """cel_reindex_static (include/cel.h): the by-action reindexing of DEVICE key bytes into DEVICE indices / offsets without
    any allocation (fixed 128 KB device scratch: n_slots <= 2^22); stream-ordered on `stream`, does not synchronise"""
    L = load_library()
    rc = L.cel_reindex_static(C.c_void_p(d_keys_ptr), int(n_slots), C.c_void_p(d_indices_ptr), C.c_void_p(d_offsets_ptr), C.c_void_p(stream))
    if rc != 0:
        raise CelError(rc, "cel_reindex_static", L.cel_strerror(rc).decode())


def workspace_bytes(n_slots, init_capacity, sort_mode):
    return int(load_library().cel_workspace_bytes(int(n_slots), int(init_capacity), int(sort_mode)))


def from_workload(w, n_slots=None, sort_mode=None, **kw):
    return Context(w.geometry, w.materials, w.physics, w.n_slots if n_slots is None else n_slots,
                   w.sort_mode if sort_mode is None else sort_mode, **kw)
