"""Far-field lower-bound queries (mcs_params.far_alpha, F1) against the EXACT oracle.

Walk-on-spheres needs a ball about the walker that lies inside the domain, not the largest one, so a
lower bound of the distance is a valid radius and the exit point keeps its distribution (harmonic measure): the
estimator is the same in expectation and in variance, only single walks differ (after their first bounded jump they
are a different realisation than the oracle's, which always jumps the exact distance).  Bars, therefore, are the
statistical ones of BASELINE.json north_star: entries within 4 Monte Carlo standard errors of the oracle's matrix
(standard error of the DIFFERENCE of two independent estimates), normalised residuals with unit variance and no
bias, the closed-form sphere spectrum, identical seeds bit-identical."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import Oracle, OracleParams, mesh_geom, steklov_eigs              # noqa: E402
from synth import box, icosphere, merge_meshes, uniform_samples, vertex_cell_samples   # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


def _cuda(a, dtype):
    return torch.as_tensor(np.ascontiguousarray(a)).to(device="cuda", dtype=dtype)


def _hit_counts(out, smp, f, K):
    """Oracle walks contributing to each entry (hat basis: vertices of the sample's face and of the exit face)."""
    rec = out["records"]
    r = rec[(rec["steps"] >= 0) & (rec["weight"] != 0)]
    vt = f[r["tri_t"]].astype(np.int64)
    vs = f[np.asarray(smp["tri"])[np.maximum(r["sample"], 0)]].astype(np.int64)
    idx = np.concatenate([vs, vt], 1)
    cnt = np.zeros((K, K), np.int64)
    seen = set()
    for p in range(6):
        for q in range(6):
            new = np.ones(len(idx), bool)
            for (p2, q2) in seen:
                new &= ~((idx[:, p2] == idx[:, p]) & (idx[:, q2] == idx[:, q]))
            np.add.at(cnt, (idx[new, p], idx[new, q]), 1)
            seen.add((p, q))
    return cnt


@pytest.mark.parametrize("exterior", [False, True])
@pytest.mark.parametrize("alpha,near", [(0.5, 4.0), (2.0, 2.0)])
def test_far_field_estimate_is_the_exact_one_in_distribution(api, exterior, alpha, near):
    v, f = merge_meshes([icosphere(2), box((0.6, 0.8, 1.0), (2, 2, 2), center=(1.9, 0.2, 0.0))])[:2]
    smp = uniform_samples(v, f, 1500, seed=21)
    W = 96
    origin = (0.1, 0.05, -0.1)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    Pf = api.Params(seed=11, walks_per_sample=W, eps=1e-3, kelvin_origin=origin, far_alpha=alpha, far_near_factor=near)
    Px = api.Params(seed=11, walks_per_sample=W, eps=1e-3, kelvin_origin=origin)
    fn = api.estimate_dtn_exterior if exterior else api.estimate_dtn_interior
    Sf, stf = fn(bvh, S, Pf, want_stats=True)
    Sx, stx = fn(bvh, S, Px, want_stats=True)
    assert torch.equal(Sf, fn(bvh, S, Pf))                                  # bit-identical run to run
    assert stf.n_far_queries > 0 and stx.n_far_queries == 0
    assert stf.n_truncated == 0 and stf.n_discarded == stx.n_discarded
    assert stf.n_steps > stx.n_steps                                         # bounded jumps are shorter: more of them
    orc = Oracle(mesh_geom(v, f))
    out = orc.estimate_dtn(OracleParams(seed=11, walks_per_sample=W, eps=1e-3, origin=origin), exterior,
                           smp["tri"], smp["bary"], smp["weight"], want_var=True)
    So, var = out["S"], out["var"]
    Sg = Sf.cpu().numpy().astype(np.float64)
    assert np.array_equal(Sg, Sg.T)
    # (a) same seed as the oracle: walks that never meet a bounded jump are the oracle's own, the others are fresh
    # realisations -- so the difference is at most that of two independent estimates (standard error sqrt(2 var)) and in
    # practice far smaller.  Entries hit by >= 200 oracle walks have a usable variance estimate: all within 4 SE; with >= 32
    # hits the weights' heavy tail shows (two independent EXACT runs put 1-2 % of such entries beyond 4 SE): <= 0.5 %.
    cnt = _hit_counts(out, smp, f, len(So))
    se = np.sqrt(2.0 * var)
    z = np.abs(Sg - So) / np.where(se > 0, se, np.inf)
    solid = (cnt >= 200) & (var > 0)
    loose = (cnt >= 32) & (var > 0)
    assert solid.sum() > 300 and loose.sum() > 1000
    assert (z[solid] > 4.0).sum() == 0, z[solid].max()
    assert (z[loose] > 4.0).sum() <= 5e-3 * loose.sum(), ((z[loose] > 4.0).sum(), loose.sum())
    assert np.linalg.norm(Sg - So) <= np.linalg.norm(np.sqrt(var))           # below one standard error in Frobenius norm
    assert np.linalg.norm(Sx.cpu().numpy() - So) <= 0.2 * np.linalg.norm(np.sqrt(var))    # the exact run: record-level parity
    if not exterior:
        assert np.abs(Sg.sum(1)).max() < 2e-5 * np.abs(Sg).max()            # annihilates constants
    # (b) independent seeds: quadratic forms x^T S x of smooth functions (sums over thousands of entries, near-Gaussian)
    # from R far-field runs against R exact runs -- same mean within 4 standard errors of the difference, same spread --
    # and the oracle's own value inside the far-field runs' spread.
    X = np.stack([v[:, 0], v[:, 1], v[:, 2], v[:, 0] * v[:, 1], v[:, 0] ** 2 - v[:, 1] ** 2, v[:, 2] ** 2,
                  np.sin(2.0 * v[:, 0]) * np.cos(v[:, 2])], 1).astype(np.float64)
    R = 8
    import dataclasses

    def forms(P):
        q = []
        for r in range(R):
            M = fn(bvh, S, dataclasses.replace(P, seed=100 + r)).cpu().numpy().astype(np.float64)
            q.append(np.einsum("vk,vw,wk->k", X, M, X))
        return np.array(q)
    qf, qx = forms(Pf), forms(Px)
    qo = np.einsum("vk,vw,wk->k", X, So, X)
    sd_f, sd_x = qf.std(0, ddof=1), qx.std(0, ddof=1)
    assert np.all(np.abs(qf.mean(0) - qx.mean(0)) <= 4.0 * np.sqrt((sd_f ** 2 + sd_x ** 2) / R)), (qf.mean(0), qx.mean(0))
    assert np.all(sd_f < 3.0 * sd_x) and np.all(sd_x < 3.0 * sd_f), (sd_f, sd_x)
    assert np.all(np.abs(qo - qf.mean(0)) <= 5.0 * sd_f), (qo, qf.mean(0), sd_f)


def test_far_field_sphere_spectrum(api):
    """Closed form: interior eigenvalues l with multiplicity 2l + 1, through the far-field estimator."""
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 8, seed=0)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    M = Oracle(mesh_geom(v, f)).mass_matrix()
    lam = {}
    for alpha in (0.0, 2.0):
        Sg, st = api.estimate_dtn_interior(bvh, S, api.Params(seed=0, walks_per_sample=128, eps=1e-3, far_alpha=alpha, far_near_factor=2.0),
                                           want_stats=True)
        lam[alpha] = steklov_eigs(Sg.cpu().numpy().astype(np.float64), M, 16)
    assert abs(lam[2.0][0]) < 1e-4
    assert np.abs(lam[2.0] - lam[0.0]).max() < 0.06
    for l, sl in ((1, slice(1, 4)), (2, slice(4, 9)), (3, slice(9, 16))):
        assert abs(lam[2.0][sl].mean() / l - 1) < 0.12, (l, lam[2.0][sl])
