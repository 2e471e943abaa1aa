"""Sparse (COO) output of the accumulation, A7 of SURVEY.md 8(a): same run sums as the dense path,
any K.  Checked against the oracle's dense accumulation (small K directly; K > 65535 on the
sub-mesh of the faces the walks touch, which is pure re-indexing)."""
import dataclasses

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import Oracle, OracleParams, mesh_geom, RECORD_DTYPE              # noqa: E402
from synth import icosphere, stress_mesh, uniform_samples, vertex_cell_samples  # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


def _cuda(a, dtype):
    return torch.as_tensor(np.ascontiguousarray(a)).to(device="cuda", dtype=dtype)


@pytest.mark.parametrize("exterior", [False, True])
def test_coo_equals_dense_upper_triangle_bitwise(api, exterior):
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 4, seed=0)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    P = api.Params(seed=2, walks_per_sample=64, eps=1e-3, include_killing=exterior, n_kill_walks=5000 if exterior else 0,
                   kelvin_origin=(0.1, 0.0, 0.05))
    dense = (api.estimate_dtn_exterior if exterior else api.estimate_dtn_interior)(bvh, S, P)
    coo, st = api.estimate_dtn_coo(bvh, S, P, exterior, want_stats=True)
    assert coo.nnz == st.n_unique and (coo.row <= coo.col).all()
    key = coo.row.long() * bvh.V + coo.col.long()
    assert (key[1:] > key[:-1]).all()                                  # sorted, one entry per (row, col)
    up = torch.triu(dense)
    if exterior:    # two passes (sample walks, then per-face killing moments): dense adds pass by pass, COO merges lists
        assert (coo.to_dense() - dense).abs().max().item() <= 2e-6 * dense.abs().max().item()
    else:
        assert torch.equal(coo.to_dense(), dense)                      # one chunk: the same sums bit for bit
    assert coo.nnz == int((up != 0).sum().item()) or coo.nnz >= int((up != 0).sum().item())
    # too small a capacity: the library says so and the binding retries
    coo2 = api.estimate_dtn_coo(bvh, S, P, exterior, capacity=100)
    assert torch.equal(coo2.val, coo.val) and torch.equal(coo2.row, coo.row) and torch.equal(coo2.col, coo.col)
    with pytest.raises(api.McsError) as e:
        api.estimate_dtn_coo(bvh, S, P, exterior, capacity=100, max_retries=1)
    assert e.value.code == api.MCS_ENOMEM


def test_coo_large_K_against_oracle_on_touched_submesh(api):
    """K = V > 65535 (no dense matrix possible with 32-bit keys): the GPU's own records are accumulated by
    the library (COO) and by the oracle on the sub-mesh of touched faces."""
    v, f, info = stress_mesh(n_faces=200_000, n_components=12, seed=5)
    assert len(v) > 65535
    smp = uniform_samples(v, f, 160, seed=1)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    P = api.Params(seed=8, walks_per_sample=16, eps=1e-3, max_steps=256)
    rec, steps = api.run_walks(bvh, S, P, False)
    coo, st = api.estimate_dtn_coo(bvh, S, P, False, want_stats=True)
    coo_b = api.estimate_dtn_coo(bvh, S, P, False)
    assert torch.equal(coo.val, coo_b.val) and torch.equal(coo.row, coo_b.row)      # bit-identical rerun
    r = rec.cpu().numpy()
    tri_t = r[:, 0].copy().view(np.int32)
    ok = tri_t >= 0
    # sub-mesh: faces touched by samples or exits, vertices renumbered
    faces_used = np.unique(np.concatenate([smp["tri"], tri_t[ok]]))
    verts_used, inv = np.unique(f[faces_used], return_inverse=True)
    f_sub = inv.reshape(-1, 3).astype(np.int32)
    face_new = -np.ones(len(f), np.int64); face_new[faces_used] = np.arange(len(faces_used))
    orec = np.zeros(len(r), RECORD_DTYPE)
    orec["sample"] = np.repeat(np.arange(len(smp["tri"])), 16)
    orec["tri_t"] = np.where(ok, face_new[np.maximum(tri_t, 0)], -1)
    orec["bary_t"][:, 1] = r[:, 1]; orec["bary_t"][:, 2] = r[:, 2]
    orec["bary_t"][:, 0] = 1.0 - r[:, 1].astype(np.float32) - r[:, 2].astype(np.float32)
    orec["weight"] = np.where(ok, r[:, 3], 0.0)
    orec["steps"] = np.where(ok, 0, -1)
    orc = Oracle(mesh_geom(v[verts_used], f_sub))
    So = orc.accumulate_hat(orec, face_new[smp["tri"]].astype(np.int32), smp["bary"])
    # scatter the GPU's COO entries into the sub-mesh numbering
    vert_new = -np.ones(len(v), np.int64); vert_new[verts_used] = np.arange(len(verts_used))
    rr, cc, vv = vert_new[coo.row.cpu().numpy()], vert_new[coo.col.cpu().numpy()], coo.val.cpu().numpy().astype(np.float64)
    assert (rr >= 0).all() and (cc >= 0).all()                         # only touched vertices appear
    Sg = np.zeros_like(So)
    Sg[rr, cc] = vv
    Sg[cc, rr] = vv
    assert np.abs(Sg - So).max() <= 3e-5 * np.abs(So).max()
    assert np.abs(Sg.sum(1)).max() < 5e-5 * np.abs(Sg).max()           # interior operator annihilates constants


def test_coo_both_operators_in_one_call_equal_the_single_calls(api):
    """mcs_estimate_dtn_both with sparse outputs: same lists as two estimate_dtn_coo calls, also after a capacity retry."""
    v, f = icosphere(3)
    smp = uniform_samples(v, f, 2001, seed=4)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    Pi = api.Params(seed=6, walks_per_sample=32, eps=1e-3)
    Pe = api.Params(seed=6, walks_per_sample=32, eps=1e-3, include_killing=True, n_kill_walks=6000, kelvin_origin=(0.1, 0.0, 0.05))
    ci = api.estimate_dtn_coo(bvh, S, Pi, False)
    ce = api.estimate_dtn_coo(bvh, S, Pe, True)
    for cap in (None, 500):
        bi, be = api.estimate_dtn_coo_both(bvh, S, Pi, Pe, capacity=cap)
        for a, b in ((bi, ci), (be, ce)):
            assert torch.equal(a.row, b.row) and torch.equal(a.col, b.col) and torch.equal(a.val, b.val)
    with pytest.raises(api.McsError) as e:
        api.estimate_dtn_coo_both(bvh, S, Pi, Pe, capacity=500, max_retries=1)
    assert e.value.code == api.MCS_ENOMEM
