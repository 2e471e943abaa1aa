"""mcs_params.nonblocking ("async on the given stream ... CUDA-graph and stream friendly"): the
dense hat-basis estimate only enqueues work -- no read-back, no allocation -- so it can be captured in a CUDA graph.
Bars: the same bits as the blocking call (same kernels, same order), eager and replayed from a graph, replay after
replay; device-side input errors, which a call that reads nothing back cannot return, turn the output into NaN."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from synth import icosphere, vertex_cell_samples          # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


def _cuda(a, dtype):
    return torch.as_tensor(np.ascontiguousarray(a)).to(device="cuda", dtype=dtype)


def _case(api, level=2, ppv=4):
    v, f = icosphere(level)
    smp = vertex_cell_samples(v, f, ppv, seed=5)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    return v, f, smp, bvh, S


def _ops(api, S, W):
    n_kill = S.n_s * W
    return ((False, api.Params(seed=7, walks_per_sample=W, eps=1e-3)),
            (True, api.Params(seed=7, walks_per_sample=W, eps=1e-3, include_killing=True, n_kill_walks=n_kill,
                              kelvin_origin=(0.1, -0.05, 0.2))))


@pytest.mark.parametrize("W", [64, 600])                  # 600 > 256: the level-1b pair merge runs too
def test_nonblocking_call_gives_the_blocking_call_bit_for_bit(api, W):
    v, f, smp, bvh, S = _case(api)
    for ext, P in _ops(api, S, W):
        fn = api.estimate_dtn_exterior if ext else api.estimate_dtn_interior
        ref, st = fn(bvh, S, P, want_stats=True)
        assert st.n_truncated == 0 and st.n_entries > 0
        ws = torch.empty(api.workspace_bytes(bvh, S, P, ext), dtype=torch.uint8, device="cuda")
        out = torch.full_like(ref, 3.0)
        fn(bvh, S, P, out=out, workspace=ws, nonblocking=True)
        torch.cuda.synchronize()
        assert torch.equal(out, ref)
        plain = fn(bvh, S, P)                              # blocking, without statistics
        assert torch.equal(plain, ref)


def test_nonblocking_call_in_a_cuda_graph(api):
    v, f, smp, bvh, S = _case(api)
    for ext, P in _ops(api, S, 128):
        fn = api.estimate_dtn_exterior if ext else api.estimate_dtn_interior
        ref = fn(bvh, S, P)
        ws = torch.empty(api.workspace_bytes(bvh, S, P, ext), dtype=torch.uint8, device="cuda")
        out = torch.zeros_like(ref)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):                          # capture_error_mode "global": a sync or an allocation would raise
            fn(bvh, S, P, out=out, workspace=ws, nonblocking=True)
        torch.cuda.synchronize()
        assert float(out.abs().sum()) == 0.0               # captured, not run
        for _ in range(3):
            out.fill_(-1.0)
            ws.random_(0, 255)                             # nothing may depend on what the workspace held
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(out, ref)


def test_nonblocking_both_operators_in_one_call_eager_and_in_a_graph(api):
    v, f, smp, bvh, S = _case(api)
    (_, Pi), (_, Pe) = _ops(api, S, 128)
    ref_i, ref_e = api.estimate_dtn_interior(bvh, S, Pi), api.estimate_dtn_exterior(bvh, S, Pe)
    ws = torch.empty(api.workspace_bytes_both(bvh, S, Pi, Pe), dtype=torch.uint8, device="cuda")
    oi, oe = torch.zeros_like(ref_i), torch.zeros_like(ref_e)
    api.estimate_dtn_both(bvh, S, Pi, Pe, out_interior=oi, out_exterior=oe, workspace=ws, nonblocking=True)
    torch.cuda.synchronize()
    assert torch.equal(oi, ref_i) and torch.equal(oe, ref_e)
    oi.zero_(); oe.zero_()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):                              # the library's two side streams fork from and join the captured stream
        api.estimate_dtn_both(bvh, S, Pi, Pe, out_interior=oi, out_exterior=oe, workspace=ws, nonblocking=True)
    torch.cuda.synchronize()
    assert float(oi.abs().sum()) == 0.0
    for _ in range(2):
        oi.fill_(-1.0); oe.fill_(-1.0)
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(oi, ref_i) and torch.equal(oe, ref_e)
    # and the ordinary call still works on the same thread's streams afterwards
    bi, be = api.estimate_dtn_both(bvh, S, Pi, Pe)
    assert torch.equal(bi, ref_i) and torch.equal(be, ref_e)


def test_nonblocking_input_errors_poison_the_output(api):
    v, f, smp, bvh, S = _case(api, level=1, ppv=2)
    K = len(v)
    out = torch.zeros((K, K), dtype=torch.float32, device="cuda")
    # a sample's face index out of range
    tri = smp["tri"].copy(); tri[3] = len(f)
    badS = api.Samples.from_arrays(tri, smp["bary"], smp["weight"])
    P = api.Params(walks_per_sample=8)
    ws = torch.empty(api.workspace_bytes(bvh, badS, P, False), dtype=torch.uint8, device="cuda")
    api.estimate_dtn_interior(bvh, badS, P, out=out, workspace=ws, nonblocking=True)
    torch.cuda.synchronize()
    assert bool(torch.isnan(out).all())
    with pytest.raises(api.McsError) as e:
        api.estimate_dtn_interior(bvh, badS, P)
    assert e.value.code == api.MCS_EINVAL
    # a vertex at the Kelvin origin (with killing walks, which must not run either)
    Pe = api.Params(walks_per_sample=8, kelvin_origin=tuple(float(x) for x in v[0]), include_killing=True, n_kill_walks=4096)
    ws = torch.empty(api.workspace_bytes(bvh, S, Pe, True), dtype=torch.uint8, device="cuda")
    out.zero_()
    api.estimate_dtn_exterior(bvh, S, Pe, out=out, workspace=ws, nonblocking=True)
    torch.cuda.synchronize()
    assert bool(torch.isnan(out).all())
    with pytest.raises(api.McsError) as e:
        api.estimate_dtn_exterior(bvh, S, Pe)
    assert e.value.code == api.MCS_EDEGENERATE
    # and a good call right after, on the same workspace, is clean
    Pg = api.Params(walks_per_sample=8, kelvin_origin=(0.0, 0.0, 0.0), include_killing=True, n_kill_walks=4096)
    good = api.estimate_dtn_exterior(bvh, S, Pg)
    api.estimate_dtn_exterior(bvh, S, Pg, out=out, workspace=ws, nonblocking=True)
    torch.cuda.synchronize()
    assert torch.equal(out, good)


def test_nonblocking_is_refused_where_the_call_has_to_read_back(api):
    v, f, smp, bvh, S = _case(api, level=1, ppv=2)
    P = api.Params(walks_per_sample=4)
    ws = torch.empty(api.workspace_bytes(bvh, S, P, False), dtype=torch.uint8, device="cuda")
    out = torch.zeros((len(v), len(v)), dtype=torch.float32, device="cuda")
    with pytest.raises(ValueError):
        api.estimate_dtn_interior(bvh, S, P, out=out, workspace=ws, nonblocking=True, want_stats=True)
    with pytest.raises(ValueError):
        api.estimate_dtn_interior(bvh, S, P, nonblocking=True)
    # straight through the C ABI: nonblocking with host_stats is MCS_EINVAL
    import ctypes as C
    cs, cb, cp = S.c(), api._basis(bvh, None), P.c()
    cp.nonblocking = 1
    m = api._Matrix(kind=0, K=len(v), dense=out.data_ptr())
    st = api.Stats()
    rc = api.lib().mcs_estimate_dtn_interior(bvh.handle, C.byref(cs), C.byref(cb), C.byref(cp), api._ptr(ws), C.c_size_t(ws.numel()),
                                             C.byref(m), C.byref(st), api._stream(bvh.device))
    assert rc == api.MCS_EINVAL
    cp.nonblocking = 2
    rc = api.lib().mcs_estimate_dtn_interior(bvh.handle, C.byref(cs), C.byref(cb), C.byref(cp), api._ptr(ws), C.c_size_t(ws.numel()),
                                             C.byref(m), None, api._stream(bvh.device))
    assert rc == api.MCS_EINVAL
