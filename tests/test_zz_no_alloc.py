"""mcs_sort_pairs_u64_static: the allocation-free entry point (workspace in a static device array of the library)
against the existing path mcs_sort_pairs_u64 (caller-provided workspace).  Integer work: the bar is bit-exact, the
same as tests/test_gpu_geometry.py::test_radix_sort_is_stable_and_exact.  Two calls in a row share the array and the
second is smaller than the first, so whatever the first one left behind is still there when it runs.

This file is named test_zz_* so that pytest collects it last (the suite runs with `pytest -x`)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as a
    a.lib()
    return a


def _case(n, bits, seed):
    rng = np.random.default_rng(seed)
    keys = rng.integers(0, 1 << min(bits, 62), size=n, dtype=np.int64)
    if n > 100:
        keys[: n // 4] = keys[n // 4: n // 4 * 2]          # many duplicates: stability is visible in the payload
    vals = np.arange(n, dtype=np.int32)
    return keys, vals


def test_static_scratch_sort_equals_the_workspace_path_on_two_calls_in_a_row(api):
    dev = torch.device("cuda:0")
    for n, bits, seed in ((700_001, 63, 1), (70_000, 17, 2)):      # several tiles + a ragged tail; then a smaller job
        keys, vals = _case(n, bits, seed)
        k_ref, v_ref = api.sort_pairs_u64(torch.from_numpy(keys).to(dev), torch.from_numpy(vals).to(dev), bits)
        k_in, v_in = torch.from_numpy(keys).to(dev), torch.from_numpy(vals).to(dev)
        torch.cuda.synchronize()
        alloc0 = torch.cuda.memory_allocated(dev)
        k, v = api.sort_pairs_u64_static(k_in, v_in, bits)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated(dev) == alloc0           # nothing through torch's allocator
        assert torch.equal(k, k_ref) and torch.equal(v, v_ref)
        order = np.argsort(keys, kind="stable")
        assert np.array_equal(k.cpu().numpy(), keys[order])
        assert np.array_equal(v.cpu().numpy(), vals[order])
        del k, v, k_in, v_in, k_ref, v_ref                          # so that the next round's allocation count starts clean


def test_static_scratch_sort_edges_and_limit(api):
    dev = torch.device("cuda:0")
    nmax = api.sort_static_max_n()
    assert nmax == 1 << 20
    for n in (0, 1):
        k, v = api.sort_pairs_u64_static(torch.arange(n, dtype=torch.int64, device=dev), torch.arange(n, dtype=torch.int32, device=dev))
        assert k.numel() == n
    # exactly the maximum works and matches the existing path
    keys, vals = _case(nmax, 40, 3)
    k_ref, v_ref = api.sort_pairs_u64(torch.from_numpy(keys).to(dev), torch.from_numpy(vals).to(dev), 40)
    k, v = api.sort_pairs_u64_static(torch.from_numpy(keys).to(dev), torch.from_numpy(vals).to(dev), 40)
    assert torch.equal(k, k_ref) and torch.equal(v, v_ref)
    # one more is refused with the clear error, inputs untouched
    keys, vals = _case(nmax + 1, 40, 4)
    k_in, v_in = torch.from_numpy(keys).to(dev), torch.from_numpy(vals).to(dev)
    with pytest.raises(api.McsError) as ei:
        api.sort_pairs_u64_static(k_in, v_in, 40)
    assert ei.value.code == -5 and "maximum" in str(ei.value)
    assert np.array_equal(k_in.cpu().numpy(), keys)
