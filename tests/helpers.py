"""Shared test helpers: golden file reader and oracle construction from a Workload."""
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def golden_values(name="survey_values.txt"):
    out = {}
    with open(os.path.join(HERE, "golden", name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v, tol = line.split()
            out[k] = (float(v), float(tol))
    return out


def make_oracle(w, n_slots=None, sort_mode=None):
    import oracle as orc
    return orc.Oracle(w.geometry, w.materials, w.physics, w.n_slots if n_slots is None else n_slots,
                      w.sort_mode if sort_mode is None else sort_mode)


def rel_close(a, b, tol):
    return abs(a - b) <= tol * max(abs(a), abs(b))
