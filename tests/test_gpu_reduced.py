"""GPU parity of the reduced Ritz-Galerkin matrix (mcs_project_galerkin; SURVEY.md 8(f)
rank 3) against the oracle, which accumulates the paper's deferred outer products D^T diag(w) D walk by walk:
(a) the projection kernels alone against fp64 Phi^T S Phi on the same S, sizes with ragged tiles;
(b) the whole path -- GPU walks, GPU nodal accumulation, GPU projection -- against the oracle's own walks and
    outer-product accumulation, within Monte Carlo standard errors (same Philox streams, fp32 against fp64)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import Oracle, OracleParams, mesh_geom                            # noqa: E402
from synth import icosphere, vertex_cell_samples                              # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


@pytest.mark.parametrize("V,K", [(1, 1), (5, 3), (64, 64), (130, 17), (642, 160), (1000, 65)])
def test_projection_kernels(api, V, K):
    rng = np.random.default_rng(V + K)
    A = rng.normal(size=(V, V)); S = (A + A.T).astype(np.float32)
    Phi = rng.normal(size=(V, K)).astype(np.float32)
    R = api.project_galerkin(torch.from_numpy(S).cuda(), torch.from_numpy(Phi).cuda())
    assert torch.equal(R, R.T)
    assert torch.equal(R, api.project_galerkin(torch.from_numpy(S).cuda(), torch.from_numpy(Phi).cuda()))
    want = Phi.astype(np.float64).T @ S.astype(np.float64) @ Phi.astype(np.float64)
    # fp32 accumulation of V (then V again) products: error ~ eps sqrt(V) |Phi|^2 |S|
    assert np.abs(R.cpu().numpy() - want).max() < 2e-6 * np.sqrt(V) * np.abs(want).max() + 1e-6


@pytest.mark.parametrize("exterior", [False, True])
def test_reduced_matrix_end_to_end_against_oracle_outer_products(api, exterior):
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 2, seed=1)
    kw = dict(seed=5, walks_per_sample=32, eps=1e-3, include_killing=exterior, n_kill_walks=2000 if exterior else 0)
    rng = np.random.default_rng(2)
    Phi = np.concatenate([np.ones((len(v), 1)), v.astype(np.float64), rng.normal(size=(len(v), 12))], 1).astype(np.float32)
    bvh = api.build_bvh(torch.from_numpy(v).cuda(), torch.from_numpy(f).cuda())
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    fn = api.estimate_dtn_exterior if exterior else api.estimate_dtn_interior
    Sg = fn(bvh, S, api.Params(**kw))
    R = api.project_galerkin(Sg, torch.from_numpy(Phi).cuda()).cpu().numpy().astype(np.float64)
    orc = Oracle(mesh_geom(v, f))
    out = orc.estimate_dtn(OracleParams(**kw), exterior, smp["tri"], smp["bary"], smp["weight"], want_var=True)
    Ro = orc.accumulate_reduced(out["records"], smp["tri"], smp["bary"], Phi.astype(np.float64))
    # same streams: the two differ by the few walks whose fp32 and fp64 paths diverge; bound by the propagated
    # standard error of the nodal entries
    se = np.sqrt(np.abs(Phi.astype(np.float64)).T ** 2 @ out["var"] @ np.abs(Phi.astype(np.float64)) ** 2)
    assert np.abs(R - Ro).max() < 0.5 * se.max() + 1e-5 * np.abs(Ro).max()
    assert np.linalg.norm(R - Ro) < 0.05 * np.linalg.norm(Ro)
    if not exterior:
        assert np.abs(R[0]).max() < 1e-5 * np.abs(R).max()                    # constants: interior kernel
        mass = 4 * np.pi / 3
        assert np.all(np.abs(np.diag(R)[1:4] / mass - 1.0) < 0.3)            # degree-1 harmonics: l = 1


@pytest.mark.parametrize("V,K,density", [(1, 1, 1.0), (37, 5, 0.3), (500, 160, 0.05), (3000, 33, 0.01), (20000, 64, 0.0005)])
def test_projection_from_coo_matches_fp64_and_dense(api, V, K, density):
    """Sorted upper-triangular COO (rows with no entries, ragged split-K chunks) against fp64, and against the dense
    kernels where V allows."""
    rng = np.random.default_rng(V)
    nnz = max(1, int(density * V * (V + 1) / 2))
    r = rng.integers(0, V, nnz); c = rng.integers(0, V, nnz)
    r, c = np.minimum(r, c), np.maximum(r, c)
    key = np.unique(r.astype(np.int64) * V + c)
    r, c = (key // V).astype(np.int32), (key % V).astype(np.int32)
    val = rng.normal(size=len(key)).astype(np.float32)
    Phi = rng.normal(size=(V, K)).astype(np.float32)
    coo = api.CooMatrix(V, torch.from_numpy(r).cuda(), torch.from_numpy(c).cuda(), torch.from_numpy(val).cuda())
    R = api.project_galerkin_coo(coo, torch.from_numpy(Phi).cuda())
    assert torch.equal(R, R.T) and torch.equal(R, api.project_galerkin_coo(coo, torch.from_numpy(Phi).cuda()))
    import scipy.sparse as sp
    U = sp.coo_matrix((val.astype(np.float64), (r, c)), shape=(V, V)).tocsr()
    Sfull = U + sp.triu(U, 1).T
    want = Phi.astype(np.float64).T @ (Sfull @ Phi.astype(np.float64))
    assert np.abs(R.cpu().numpy() - want).max() < 3e-6 * np.sqrt(len(key) + 1) * max(np.abs(want).max(), 1e-3) / max(np.sqrt(K), 1) + 1e-5
    if V <= 3000:
        Rd = api.project_galerkin(torch.from_numpy(Sfull.toarray().astype(np.float32)).cuda(), torch.from_numpy(Phi).cuda())
        assert (R - Rd).abs().max().item() < 1e-4 * max(np.abs(want).max(), 1e-3)
    bad = api.CooMatrix(V, coo.col.clone(), coo.row.clone(), coo.val)           # lower triangle: rejected
    if (r != c).any():
        with pytest.raises(api.McsError):
            api.project_galerkin_coo(bad, torch.from_numpy(Phi).cuda())


def test_reduced_matrix_from_sparse_estimate(api):
    """estimate_dtn_coo -> project_galerkin_coo equals estimate (dense) -> project_galerkin on the same walks."""
    v, f = icosphere(3)
    smp = vertex_cell_samples(v, f, 1, seed=4)
    bvh = api.build_bvh(torch.from_numpy(v).cuda(), torch.from_numpy(f).cuda())
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    P = api.Params(seed=3, walks_per_sample=32, eps=1e-3)
    Phi = torch.from_numpy(np.random.default_rng(0).normal(size=(len(v), 40)).astype(np.float32)).cuda()
    Rd = api.project_galerkin(api.estimate_dtn_interior(bvh, S, P), Phi)
    Rc = api.project_galerkin_coo(api.estimate_dtn_coo(bvh, S, P, exterior=False), Phi)
    assert (Rd - Rc).abs().max().item() < 2e-5 * Rd.abs().max().item()
