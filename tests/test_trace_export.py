"""Chrome-trace export of the device-side timeline: formatting only, no GPU."""
import json

import numpy as np

from paper_2503_17608_b200 import trace_export as T


def test_chrome_trace_structure():
    names = ["fill_sort", "scatter", "charged", "push"]
    never = np.iinfo(np.uint64).max
    stamps = np.zeros((3, 4, 2), np.uint64)
    stamps[:, :, 0] = never
    t = 1_000_000
    for k in range(2):                       # iteration 2 never ran
        for j in (0, 1, 3):                  # "charged" did not run
            stamps[k, j] = (t, t + 2000)
            t += 3000
    counts = np.array([[0, 0, 1, 2, 3, 0, 0, 10], [1, 0, 0, 2, 2, 1, 0, 10], [0] * 8], np.uint32)
    tr = T.chrome_trace(names, stamps, counts)
    json.dumps(tr)                           # serialisable
    x = [e for e in tr["traceEvents"] if e["ph"] == "X"]
    assert len(x) == 6 and all(e["dur"] == 2.0 for e in x)
    assert x[0]["ts"] == 0.0 and x[1]["ts"] == 3.0 and {e["name"] for e in x} == {"fill_sort", "scatter", "push"}
    c = [e for e in tr["traceEvents"] if e["ph"] == "C" and e["name"] == "tracks"]
    assert [e["args"]["alive"] for e in c] == [6, 6]
    rows = T.summary_rows(names, stamps, counts, every=1)
    assert len(rows) == 3 and "charged" not in rows[0]


def test_empty_trace():
    tr = T.chrome_trace(["a"], np.zeros((0, 1, 2), np.uint64), np.zeros((0, 8), np.uint32))
    assert tr["traceEvents"] == []
