"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol include/cel.h
declares; struct layouts match the header; the workload generators are deterministic."""
import ctypes as C
import os
import re

import numpy as np

from paper_2503_17608_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    from paper_2503_17608_b200 import build, binding
    build.build()
    L = binding.load_library()
    header = open(os.path.join(ROOT, "include", "cel.h")).read()
    declared = set(re.findall(r"\b(cel_[a-z_]+)\s*\(", header))
    declared -= {"cel_ctx"}
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name
    # error strings are served without a device
    assert L.cel_strerror(0) == b"ok" and L.cel_strerror(-4) == b"initializer stack overflow"
    # workspace size is pure host arithmetic
    n = binding.workspace_bytes(1 << 20, 1 << 24, 1)
    assert n > (1 << 20) * (64 + 128 + 4 + 2) + (1 << 24) * 64  # state + secondary staging + index + key bytes, stack


def test_struct_layouts_match_header():
    from paper_2503_17608_b200 import binding
    assert binding.PRIMARY_DTYPE.itemsize == 64 and binding.TRACK_DTYPE.itemsize == 80
    assert C.sizeof(binding.cel_material) == 24
    assert C.sizeof(binding.cel_physics) == 56
    assert C.sizeof(binding.cel_geometry) == 8 + 24 + 24 + 24


def test_create_fails_loudly_without_gpu():
    import pytest
    import torch
    from paper_2503_17608_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    w = W.config1(n_events=2, n_slots=64)
    with pytest.raises(binding.CelError) as ei:
        binding.from_workload(w)
    assert ei.value.code == -2      # CEL_ERR_CUDA: no CPU fallback


def test_workloads_are_seeded_and_shaped():
    a = W.config4(); b = W.config4()
    assert np.array_equal(a.primaries, b.primaries)
    assert len(a.primaries) == 5000 and a.n_slots == 1 << 22
    assert np.all((a.primaries["energy"] >= 1e3) & (a.primaries["energy"] <= 1e5))
    assert np.allclose(np.linalg.norm(a.primaries["dir"], axis=1), 1.0, atol=1e-15)
    eta = -np.log(np.tan(0.5 * np.arccos(a.primaries["dir"][:, 2])))
    assert np.abs(eta).max() <= 2.5 + 1e-9
    assert (a.primaries["ptype"] == 0).sum() == 2500
    g = a.geometry
    assert len(g["vol_material"]) == 24 and g["vol_bin"].max() == 11
    c = W.config2()
    assert len(c.geometry["bounds"]) == 101 and abs(c.geometry["bounds"][-1] - 40.0) < 1e-12
    assert W.config5().n_events == 2000 and W.config3().geometry["field"][0] == 1.0
