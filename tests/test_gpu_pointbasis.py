"""GPU parity of the point-based k-NN bilateral basis (mcs_basis.kind 1; App. B, Eq. 44-45; SURVEY.md 8(f)
rank 1) against the oracle: neighbours bit-exact on tie-free queries, weights to fp32 accuracy, and the assembled
matrices within 4 Monte Carlo standard errors; bit-identical reruns, exact symmetry, zero row sums."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import Oracle, OracleParams, mesh_geom                            # noqa: E402
from oracle import PointBasis as OrcPointBasis                                 # noqa: E402
from synth import (box, fps_samples, icosphere, merge_meshes, stress_mesh, torus, uniform_samples,   # noqa: E402
                   vertex_cell_samples)


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


def _cuda(a, dtype):
    return torch.as_tensor(np.ascontiguousarray(a)).to(device="cuda", dtype=dtype)


def _points_on(v, f, n, seed):
    """Point cloud = farthest-point samples of the surface with their face normals (R3 of SURVEY.md 8(c))."""
    smp = fps_samples(v, f, n, n_candidates=max(20 * n, 4000), seed=seed)
    tv = v[f[smp["tri"]]].astype(np.float64)
    p = np.einsum("qk,qkd->qd", smp["bary"].astype(np.float64), tv)
    nrm = np.cross(tv[:, 1] - tv[:, 0], tv[:, 2] - tv[:, 0])
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    return p.astype(np.float32), nrm.astype(np.float32), smp


@pytest.mark.parametrize("k", [1, 8, 16])
def test_knn_weights_match_oracle(api, k):
    v, f = merge_meshes([icosphere(3), torus(1.0, 0.3, 40, 20, axis="z", center=(0, 0, 2.5))])[:2]
    pts, nrm, _ = _points_on(v, f, 700, seed=1)
    sigma = 0.12
    rng = np.random.default_rng(k)
    q = (pts[rng.integers(0, len(pts), 3000)] + rng.normal(scale=0.05, size=(3000, 3))).astype(np.float32)
    nq = rng.normal(size=(3000, 3)); nq /= np.linalg.norm(nq, axis=1, keepdims=True)
    nq = nq.astype(np.float32)
    idx_o, w_o = Oracle(mesh_geom(v, f)).knn_weights(OrcPointBasis(pts, nrm, k=k, sigma=sigma, tau_n=0.8), q, nq)
    pb = api.PointBasis.from_arrays(pts, nrm, k=k, sigma=sigma, tau_n=0.8)
    idx_g, w_g = api.knn_weights(pb, _cuda(q, torch.float32), _cuda(nq, torch.float32))
    idx_g, w_g = idx_g.cpu().numpy(), w_g.cpu().numpy()
    # tie-free: consecutive neighbour distances (and the first one left out) differ by more than fp32 rounding
    d2 = ((q[:, None, :].astype(np.float64) - pts[None].astype(np.float64)) ** 2).sum(2)
    ds = np.sort(d2, axis=1)[:, :k + 1]
    keep = (np.diff(ds, axis=1) > 1e-5 * ds[:, 1:]).all(1)
    assert keep.mean() > 0.9
    assert np.array_equal(idx_g[keep], idx_o[keep])                    # same neighbours in the same order
    assert np.abs(w_g[keep] - w_o[keep]).max() < 2e-5
    assert np.abs(w_g.sum(1) - 1).max() < 1e-5 and (w_g >= 0).all()


def test_knn_more_neighbours_than_points_and_errors(api):
    pts = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0]], np.float32)
    nrm = np.tile([0, 0, 1], (3, 1)).astype(np.float32)
    pb = api.PointBasis.from_arrays(pts, nrm, k=8, sigma=1.0)
    idx, w = api.knn_weights(pb, _cuda([[0.1, 0.1, 0.0]], torch.float32), _cuda([[0, 0, 1]], torch.float32))
    assert idx[0, :3].tolist() == [0, 1, 2] and (idx[0, 3:] == -1).all() and abs(w[0, :3].sum().item() - 1) < 1e-6
    for bad in (dict(k=0), dict(k=17), dict(sigma=0.0), dict(tau_n=0.0)):
        with pytest.raises(api.McsError):
            api.knn_weights(api.PointBasis.from_arrays(pts, nrm, **bad), _cuda([[0, 0, 0]], torch.float32), _cuda([[0, 0, 1]], torch.float32))


@pytest.mark.parametrize("exterior", [False, True])
def test_point_basis_matrix_matches_oracle(api, exterior):
    """Icosphere L3, 400 FPS points as the function space, quadrature samples on the vertex cells."""
    v, f = icosphere(3)
    pts, nrm, _ = _points_on(v, f, 400, seed=2)
    smp = vertex_cell_samples(v, f, 2, seed=0)
    sigma = 0.5 * float(np.sqrt(4 * np.pi / 400))
    kw = dict(seed=9, walks_per_sample=64, eps=1e-3, include_killing=exterior, n_kill_walks=40_000 if exterior else 0)
    origin = (0.1, 0.0, -0.05)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    pb = api.PointBasis.from_arrays(pts, nrm, k=8, sigma=sigma, tau_n=0.8)
    fn = api.estimate_dtn_exterior if exterior else api.estimate_dtn_interior
    A, st = fn(bvh, S, api.Params(kelvin_origin=origin, **kw), want_stats=True, basis=pb)
    assert A.shape == (400, 400) and torch.equal(A, A.T)
    assert torch.equal(A, fn(bvh, S, api.Params(kelvin_origin=origin, **kw), basis=pb))         # bit-identical rerun
    Sg = A.cpu().numpy().astype(np.float64)
    orc = Oracle(mesh_geom(v, f))
    out = orc.estimate_dtn_points(OrcPointBasis(pts, nrm, k=8, sigma=sigma, tau_n=0.8), OracleParams(origin=origin, **kw),
                                  exterior, smp["tri"], smp["bary"], smp["weight"], want_var=True)
    So, var = out["S"], out["var"]
    assert np.linalg.norm(Sg - So) <= np.linalg.norm(np.sqrt(var))       # same streams: far below the MC error
    se = np.sqrt(2.0 * var)
    big = var > np.quantile(var[var > 0], 0.5)                           # entries with a meaningful variance estimate
    bad = (np.abs(Sg - So) > 4.0 * se + 2e-6 * np.abs(So).max()) & big
    assert bad.sum() <= max(1, int(1e-3 * big.sum())), (bad.sum(), big.sum())
    if not exterior:
        assert np.abs(Sg.sum(1)).max() < 5e-5 * np.abs(Sg).max()          # partition of unity: constants annihilated
    assert np.linalg.eigvalsh(Sg).min() > -1e-5 * np.abs(Sg).max()
    # the library's accumulation of its own records equals the oracle's accumulation of them
    rec, steps = api.run_walks(bvh, S, api.Params(kelvin_origin=origin, **kw), exterior)
    from oracle import RECORD_DTYPE
    r = rec.cpu().numpy()
    tri_t = r[:, 0].copy().view(np.int32)
    ok = tri_t >= 0
    n_main = len(smp["tri"]) * 64
    orec = np.zeros(len(r), RECORD_DTYPE)
    orec["sample"] = np.where(np.arange(len(r)) < n_main, np.arange(len(r)) // 64, -1)
    orec["tri_t"] = tri_t
    bt = np.stack([1.0 - r[:, 1] - r[:, 2], r[:, 1], r[:, 2]], 1).astype(np.float64)
    orec["t"] = np.where(ok[:, None], np.einsum("qk,qkd->qd", bt, v[f[np.maximum(tri_t, 0)]].astype(np.float64)), 0.0)
    orec["weight"] = np.where(ok, r[:, 3], 0.0)
    orec["steps"] = np.where(ok, 0, -1)
    S2 = orc.accumulate_points(OrcPointBasis(pts, nrm, k=8, sigma=sigma, tau_n=0.8), orec, smp["tri"], smp["bary"], smp["weight"])
    assert np.abs(Sg - S2).max() <= 5e-5 * np.abs(S2).max()


def test_point_basis_stress_mesh_config4_style(api):
    """BASELINE config 4's shape of problem on one mesh: 512 FPS samples that are also the nodes of the function
    space, 64 walks each, on a 20k-face stress mesh (slivers, duplicates, flips)."""
    v, f, info = stress_mesh(n_faces=20_000, n_components=8, seed=4)
    pts, nrm, smp = _points_on(v, f, 512, seed=3)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    pb = api.PointBasis.from_arrays(pts, nrm, k=8, sigma=0.15, tau_n=0.8)
    P = api.Params(seed=2, walks_per_sample=64, eps=1e-3, max_steps=512)
    A, st = api.estimate_dtn_interior(bvh, S, P, want_stats=True, basis=pb)
    assert torch.equal(A, api.estimate_dtn_interior(bvh, S, P, basis=pb)) and torch.equal(A, A.T)
    Sg = A.cpu().numpy().astype(np.float64)
    assert np.abs(Sg.sum(1)).max() < 1e-4 * np.abs(Sg).max()
    assert np.linalg.eigvalsh(Sg).min() > -1e-5 * np.abs(Sg).max()
    out = Oracle(mesh_geom(v, f)).estimate_dtn_points(OrcPointBasis(pts, nrm, k=8, sigma=0.15, tau_n=0.8),
                                                      OracleParams(seed=2, walks_per_sample=64, eps=1e-3, max_steps=512),
                                                      False, smp["tri"], smp["bary"], smp["weight"], want_var=True)
    assert np.linalg.norm(Sg - out["S"]) <= np.linalg.norm(np.sqrt(out["var"]))
    with pytest.raises(api.McsError):                                   # sparse output / Alg. 1 not offered for this basis
        api.estimate_dtn_interior(bvh, S, api.Params(walks_per_sample=2, estimator=1, inset=0.01), basis=pb)


def test_knn_grid_path_matches_oracle_and_exhaustive(api):
    """K > 1024: the neighbour search runs through the uniform grid.  Same neighbours and weights as the oracle's
    exhaustive search on tie-free queries, including queries far outside the points' bounding box."""
    v, f = merge_meshes([icosphere(4), torus(1.0, 0.3, 80, 40, axis="z", center=(0, 0, 2.5))])[:2]
    pts, nrm, _ = _points_on(v, f, 5000, seed=5)
    k, sigma = 8, 0.05
    rng = np.random.default_rng(7)
    q = np.concatenate([pts[rng.integers(0, len(pts), 4000)] + rng.normal(scale=0.02, size=(4000, 3)),
                        rng.uniform(-6, 6, size=(300, 3))]).astype(np.float32)
    nq = rng.normal(size=(len(q), 3)); nq /= np.linalg.norm(nq, axis=1, keepdims=True)
    nq = nq.astype(np.float32)
    idx_o, w_o = Oracle(mesh_geom(v, f)).knn_weights(OrcPointBasis(pts, nrm, k=k, sigma=sigma, tau_n=0.8), q, nq)
    pb = api.PointBasis.from_arrays(pts, nrm, k=k, sigma=sigma, tau_n=0.8)
    idx_g, w_g = api.knn_weights(pb, _cuda(q, torch.float32), _cuda(nq, torch.float32))
    idx_g, w_g = idx_g.cpu().numpy(), w_g.cpu().numpy()
    d2 = ((q[:, None, :].astype(np.float64) - pts[None].astype(np.float64)) ** 2).sum(2)
    ds = np.sort(d2, axis=1)[:, :k + 1]
    keep = (np.diff(ds, axis=1) > 1e-5 * ds[:, 1:]).all(1)
    assert keep.mean() > 0.9
    assert np.array_equal(idx_g[keep], idx_o[keep])
    near = np.arange(len(q)) < 4000
    assert np.abs(w_g[keep & near] - w_o[keep & near]).max() < 5e-5
    # queries 100 sigma away: the exponents are ~1e4 and their fp32 rounding shows in the weights
    assert np.abs(w_g[keep & ~near] - w_o[keep & ~near]).max() < 5e-3
    assert np.abs(w_g.sum(1) - 1).max() < 1e-5


def test_point_basis_matrix_grid_path(api):
    """The estimator with K = 3000 nodes (grid search inside the accumulation) against the oracle."""
    v, f = icosphere(4)
    pts, nrm, _ = _points_on(v, f, 3000, seed=6)
    smp = vertex_cell_samples(v, f, 1, seed=0)
    sigma = 0.5 * float(np.sqrt(4 * np.pi / 3000))
    kw = dict(seed=4, walks_per_sample=16, eps=1e-3)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    pb = api.PointBasis.from_arrays(pts, nrm, k=8, sigma=sigma, tau_n=0.8)
    A = api.estimate_dtn_interior(bvh, S, api.Params(**kw), basis=pb)
    assert torch.equal(A, api.estimate_dtn_interior(bvh, S, api.Params(**kw), basis=pb)) and torch.equal(A, A.T)
    Sg = A.cpu().numpy().astype(np.float64)
    out = Oracle(mesh_geom(v, f)).estimate_dtn_points(OrcPointBasis(pts, nrm, k=8, sigma=sigma, tau_n=0.8), OracleParams(**kw),
                                                      False, smp["tri"], smp["bary"], smp["weight"], want_var=True)
    assert np.linalg.norm(Sg - out["S"]) <= np.linalg.norm(np.sqrt(out["var"]))
    assert np.abs(Sg.sum(1)).max() < 5e-5 * np.abs(Sg).max()


def test_point_basis_both_operators_in_one_call(api):
    """mcs_estimate_dtn_both with the k-NN point basis: the overlapped call equals the two single calls bit for bit."""
    v, f = merge_meshes([icosphere(3), box((0.7, 0.5, 0.9), (4, 4, 4), center=(2.4, 0.0, 0.1))])[:2]
    pts, nrm, _ = _points_on(v, f, 300, seed=5)
    smp = uniform_samples(v, f, 900, seed=6)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    pb = api.PointBasis.from_arrays(pts, nrm, k=8, sigma=0.1, tau_n=0.8)
    Pi = api.Params(seed=3, walks_per_sample=32, eps=1e-3)
    Pe = api.Params(seed=3, walks_per_sample=32, eps=1e-3, include_killing=True, n_kill_walks=3000, kelvin_origin=(0.05, 0.0, 0.02))
    Ai = api.estimate_dtn_interior(bvh, S, Pi, basis=pb).clone()
    Ae = api.estimate_dtn_exterior(bvh, S, Pe, basis=pb).clone()
    Bi, Be = api.estimate_dtn_both(bvh, S, Pi, Pe, basis=pb)
    assert Bi.shape == (300, 300) and torch.equal(Bi, Ai) and torch.equal(Be, Ae)
