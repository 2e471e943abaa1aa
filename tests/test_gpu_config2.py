"""BASELINE config 2 at FULL size (Fig. 3/7): two level-5 icospheres
(10 242 vertices each) with centres 2.5 apart plus the 40 000-face torus between them (axis along x),
V = 40 484, 2048 walks per vertex = 8 sample points x 256 walks = 82.9 M walks per operator, sparse output.
The closed-form variant 2a (spheres only: capacity, decay over distance) is in test_gpu_estimator.py; here the
block structure of the operators (SURVEY.md 8(c) "Coupling (config 2b)"): the interior operator does not couple
disconnected solids, the exterior one does, with the torus in between."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from synth import two_spheres_torus_scene, vertex_cell_samples                # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


def test_config2b_full_size_block_structure(api):
    v, f, vid, fid = two_spheres_torus_scene(level=5, distance=2.5, with_torus=True)
    assert len(v) == 40_484 and len(f) == 80_960
    smp = vertex_cell_samples(v, f, 8, seed=0)
    W = 256
    assert len(smp["tri"]) * W == 40_484 * 2048
    bvh = api.build_bvh(torch.as_tensor(v).cuda(), torch.as_tensor(f).cuda())
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    comp = torch.as_tensor(vid).cuda().long()
    origin = (-1.25, 0.0, 0.0)                                       # centre of the first sphere (the torus centre is in its hole)
    Pi = api.Params(seed=0, walks_per_sample=W, eps=1e-3)
    Pe = api.Params(seed=0, walks_per_sample=W, eps=1e-3, kelvin_origin=origin)
    ci, sti = api.estimate_dtn_coo(bvh, S, Pi, False, want_stats=True)
    ce, ste = api.estimate_dtn_coo(bvh, S, Pe, True, want_stats=True)
    assert sti.n_walks == 40_484 * 2048 and sti.n_truncated == 0 and ste.n_truncated == 0
    assert sti.n_discarded == 0 and ste.n_discarded == 0
    # interior: a walk never leaves its solid, so no entry joins two components -- exactly, not statistically
    assert bool((comp[ci.row.long()] == comp[ci.col.long()]).all())
    # exterior: every pair of components is coupled through the ambient space
    cr, cc = comp[ce.row.long()], comp[ce.col.long()]
    val = ce.val.double()
    fro = {}
    for a in range(3):
        for b in range(a, 3):
            m = ((cr == a) & (cc == b)) | ((cr == b) & (cc == a))
            fro[(a, b)] = float(torch.sqrt((val[m] ** 2).sum()).item())
            assert int(m.sum().item()) > 0
    assert fro[(0, 1)] > 0 and fro[(0, 2)] > 0 and fro[(1, 2)] > 0
    # sphere-torus (gap 0.3) couples more strongly than sphere-sphere (gap 0.5, the torus tube partly in between)
    assert fro[(0, 2)] > fro[(0, 1)] and fro[(1, 2)] > fro[(0, 1)]
    assert fro[(0, 1)] < 0.2 * min(fro[(0, 0)], fro[(1, 1)])
    # both operators without the killing term annihilate constants (footnote at PAPER.md:385): row sums of the full
    # symmetric matrix from its upper triangle
    for coo in (ci, ce):
        rs = torch.zeros(len(v), dtype=torch.float64, device="cuda")
        rs.index_add_(0, coo.row.long(), coo.val.double())
        off = coo.row != coo.col
        rs.index_add_(0, coo.col.long()[off], coo.val.double()[off])
        assert rs.abs().max().item() < 2e-4 * coo.val.abs().max().item()
    # the two operators in one call, bit-identical to the single calls (schedule independence at 83 M walks each)
    bi, be = api.estimate_dtn_coo_both(bvh, S, Pi, Pe, capacity=max(ci.nnz, ce.nnz) + 1024)
    assert torch.equal(bi.val, ci.val) and torch.equal(bi.row, ci.row) and torch.equal(bi.col, ci.col)
    assert torch.equal(be.val, ce.val) and torch.equal(be.row, ce.row) and torch.equal(be.col, ce.col)
