"""cel_reindex_static (include/cel.h; paper_2503_17608_b200/csrc/cel_noalloc.cu): the by-action reindexing of one step
iteration (S2) with its scratch in a fixed file-scope device array, for callers that may not allocate.
Checked against the existing path — the index array and offsets the transport's own sort (k_fill_sort) produces on the
debug surface — bit for bit (integer work: no tolerance), on two calls in a row that share the scratch array.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_2503_17608_b200 import workloads as W

pytestmark = pytest.mark.gpu

VACANT = 7


@pytest.fixture(scope="module")
def binding():
    import torch
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    from paper_2503_17608_b200 import build, binding as b
    build.build()
    b.load_library()
    return b


def static_reindex(binding, keys):
    """host key bytes -> device, cel_reindex_static on torch's current stream, results back on the host"""
    import torch
    dev = torch.device("cuda", 0)
    n = len(keys)
    d_keys = torch.from_numpy(np.ascontiguousarray(keys, dtype=np.uint8)).to(dev) if n else torch.empty(4, dtype=torch.uint8, device=dev)
    # outputs pre-filled with a pattern: every entry must be written by the call
    d_idx = torch.full((max(n, 1),), 0x7fffffff, dtype=torch.int32, device=dev)
    d_off = torch.full((9,), 0x7fffffff, dtype=torch.int32, device=dev)
    binding.reindex_static(d_keys.data_ptr(), n, d_idx.data_ptr(), d_off.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return d_idx.cpu().numpy().view(np.uint32)[:n], d_off.cpu().numpy().view(np.uint32)


def existing_path_pairs(binding, w, n_pairs):
    """(keys the transport's sort saw, its index array, its offsets) for n_pairs consecutive iterations. With no secondaries
    (config 1: photons, electrons deposited locally) the stack is empty after the first fill, so the actions of the state
    after iteration k are exactly the keys iteration k+1 sorts."""
    ctx = binding.from_workload(w)
    ctx.begin(w.primaries, w.n_events)
    ctx.step()
    out = []
    for _ in range(n_pairs):
        assert len(ctx.initializers()) == 0
        keys = ctx.state()["action"].astype(np.uint8)
        ctx.step()
        idx, off = ctx.indices()
        out.append((keys, idx.copy(), off.copy()))
    ctx.close()
    return out


def test_static_reindex_equals_existing_path_twice(binding):
    # 30 tiles with a ragged last one; photoelectric, Compton, photon moves and vacancies
    w = W.config1(n_events=25000, n_slots=30000 + 77)
    pairs = existing_path_pairs(binding, w, 2)
    assert not np.array_equal(pairs[0][0], pairs[1][0])          # two different key arrays
    for keys, ref_idx, ref_off in pairs:                         # two calls in a row on the shared scratch
        assert len(np.unique(keys)) >= 3 and (keys == VACANT).any()
        idx, off = static_reindex(binding, keys)
        assert np.array_equal(off, ref_off)
        assert np.array_equal(idx, ref_idx)                      # the whole permutation, vacant tail included


def test_static_reindex_all_keys_and_stale_scratch(binding):
    """all 8 keys, first a large call and then smaller ones (rows of the higher tiles keep the large call's counts and must
    not be read), against the definition: a stable sort of the slots by key"""
    rng = np.random.default_rng(17608)
    for n in (binding.reindex_static_max_slots(), 1 << 20, 5000 + 3, 1024, 1, 0):
        keys = rng.integers(0, 8, size=n, dtype=np.uint8) | (rng.integers(0, 3, size=n, dtype=np.uint8) << 4)   # (ptype bits ignored)
        idx, off = static_reindex(binding, keys)
        k = keys & 7
        assert np.array_equal(idx, np.argsort(k, kind="stable").astype(np.uint32))
        assert np.array_equal(off, np.concatenate([[0], np.cumsum(np.bincount(k, minlength=8))]).astype(np.uint32))


def test_static_reindex_rejects_what_the_scratch_cannot_hold(binding):
    import torch
    buf = torch.zeros(16, dtype=torch.int32, device="cuda:0")
    with pytest.raises(binding.CelError) as ei:
        binding.reindex_static(buf.data_ptr(), binding.reindex_static_max_slots() + 1, buf.data_ptr(), buf.data_ptr(), 0)
    assert ei.value.code == -11 and "static scratch" in str(ei.value)       # CEL_ERR_TOO_LARGE, nothing launched
    with pytest.raises(binding.CelError) as ei:
        binding.reindex_static(buf.data_ptr() + 1, 8, buf.data_ptr(), buf.data_ptr(), 0)   # misaligned keys
    assert ei.value.code == -1
    torch.cuda.synchronize()
