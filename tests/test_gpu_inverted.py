"""GPU parity of the exact Kelvin-inverted-face query (mcs_params.exterior_query = 1; reading E4; the paper's
"spherical-triangular elements ... (non-planar) distance queries") against the oracle's E4 walks (fp64,
brute force over all faces with the closed form): records walk for walk on the same Philox streams, the matrix within
the Monte Carlo error, and the cross-check SURVEY.md 8(f) rank 4 asks for -- against the conservative-radius walks (E3)
the exact query takes fewer, longer jumps and estimates the same matrix."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import Oracle, OracleParams, mesh_geom                            # noqa: E402
from synth import icosphere, merge_meshes, stress_mesh, torus, uniform_samples, vertex_cell_samples   # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


def _scene():
    parts = [icosphere(3, 1.0, (-1.25, 0, 0)), icosphere(3, 1.0, (1.25, 0, 0)), torus(1.0, 0.3, 40, 20, axis="x")]
    v, f, _, _ = merge_meshes(parts)
    return v, f, (-1.25, 0.1, 0.05)


CASES = {
    "icosphere3": lambda: (*icosphere(3), (0.2, -0.1, 0.15)),
    "scene": _scene,
}


@pytest.mark.parametrize("name", list(CASES))
def test_exact_inverted_walks_match_the_oracle(api, name):
    v, f, origin = CASES[name]()
    smp = uniform_samples(v, f, 300, seed=3)
    bvh = api.build_bvh(torch.as_tensor(v).cuda(), torch.as_tensor(f).cuda())
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    W = 32
    kw = dict(seed=5, walks_per_sample=W, eps=1e-3, include_killing=True, n_kill_walks=2000)
    P = api.Params(kelvin_origin=origin, exterior_query=1, **kw)
    rec, steps, st = api.run_walks(bvh, S, P, True, want_stats=True)
    rec2, steps2 = api.run_walks(bvh, S, P, True)
    assert torch.equal(rec.view(torch.int32), rec2.view(torch.int32)) and torch.equal(steps, steps2)
    rec, steps = rec.cpu().numpy(), steps.cpu().numpy()
    orc = Oracle(mesh_geom(v, f))
    orec, _ = orc.run_walks(OracleParams(origin=origin, exterior_query=1, **kw), True, smp["tri"], smp["bary"], smp["weight"])
    assert st.n_truncated == int((orec["steps"] == -3).sum() + (orec["steps"] == -1).sum()) or abs(st.n_truncated - int((orec["steps"] < -0).sum())) <= 4
    same = steps == orec["steps"]
    assert same.mean() >= 0.95, same.mean()
    ok = same & (steps >= 0)
    tri_t = rec[:, 0].copy().view(np.int32)
    assert (tri_t[ok] == orec["tri_t"][ok]).mean() > 0.95
    bt = np.stack([1 - rec[:, 1] - rec[:, 2], rec[:, 1], rec[:, 2]], 1).astype(np.float64)
    t_gpu = np.einsum("qk,qkd->qd", bt[ok], v[f[tri_t[ok]]].astype(np.float64))
    err = np.linalg.norm(t_gpu - orec["t"][ok], axis=1)
    assert np.quantile(err, 0.98) < 5e-4 and np.median(err) < 2e-5, np.quantile(err, [0.5, 0.98, 1.0])
    rel = np.abs(rec[ok, 3] - orec["weight"][ok]) / np.abs(orec["weight"][ok]).max()
    assert np.quantile(rel, 0.98) < 2e-4
    # against the conservative radius E3 on the same samples: fewer jumps, never more queries' worth of walk
    P3 = api.Params(kelvin_origin=origin, **kw)
    _, steps3, st3 = api.run_walks(bvh, S, P3, True, want_stats=True)
    assert st.n_steps < 0.95 * st3.n_steps, (st.n_steps, st3.n_steps)


def test_exact_inverted_matrix_against_oracle_and_against_the_conservative_radius(api):
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 4, seed=0)
    origin = (0.25, 0.1, -0.15)
    bvh = api.build_bvh(torch.as_tensor(v).cuda(), torch.as_tensor(f).cuda())
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    kw = dict(seed=4, walks_per_sample=96, eps=1e-3, include_killing=True, n_kill_walks=40_000)
    A4 = api.estimate_dtn_exterior(bvh, S, api.Params(kelvin_origin=origin, exterior_query=1, **kw))
    assert torch.equal(A4, api.estimate_dtn_exterior(bvh, S, api.Params(kelvin_origin=origin, exterior_query=1, **kw)))
    assert torch.equal(A4, A4.T)
    A3 = api.estimate_dtn_exterior(bvh, S, api.Params(kelvin_origin=origin, **kw))
    orc = Oracle(mesh_geom(v, f))
    out = orc.estimate_dtn(OracleParams(origin=origin, exterior_query=1, **kw), True, smp["tri"], smp["bary"], smp["weight"], want_var=True)
    S4 = A4.cpu().numpy().astype(np.float64)
    se = np.linalg.norm(np.sqrt(out["var"]))
    assert np.linalg.norm(S4 - out["S"]) <= se                          # same streams: far closer than the Monte Carlo error
    se_e = np.sqrt(np.maximum(out["var"], 0))
    bad = np.abs(S4 - out["S"]) > 4 * se_e + 2e-6 * np.abs(out["S"]).max()
    assert bad.sum() <= max(1, int(1e-4 * bad.size))
    S3 = A3.cpu().numpy().astype(np.float64)
    assert np.linalg.norm(S4 - S3) <= 2.5 * se                          # two estimates of the same matrix (independent walks)
    cap4, cap3 = S4.sum() / (4 * np.pi), S3.sum() / (4 * np.pi)         # capacity of the (faceted) unit sphere
    assert abs(cap4 - cap3) < 0.02 and 0.95 < cap4 < 1.01


def test_exact_inverted_query_rejects_what_it_does_not_cover(api):
    v, f = icosphere(1)
    smp = uniform_samples(v, f, 8, seed=0)
    bvh = api.build_bvh(torch.as_tensor(v).cuda(), torch.as_tensor(f).cuda())
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    for bad, ext in ((api.Params(walks_per_sample=4, exterior_query=1), False),
                     (api.Params(walks_per_sample=4, exterior_query=1, far_alpha=0.5), True),
                     (api.Params(walks_per_sample=4, exterior_query=2), True)):
        with pytest.raises(api.McsError) as e:
            api.run_walks(bvh, S, bad, ext)
        assert e.value.code == api.MCS_EINVAL


def test_exact_inverted_walks_on_a_stress_mesh(api):
    """In-the-wild style mesh (slivers, duplicates, many components; sidedness repaired first): E4 walks against the
    oracle on a sample subset, and the step count against E3."""
    v, f, info = stress_mesh(n_faces=30_000, n_components=7, seed=9)
    from synth import fps_samples
    smp = fps_samples(v, f, 400, n_candidates=8000, seed=1)
    bvh = api.build_bvh(torch.as_tensor(v).cuda(), torch.as_tensor(f).cuda())
    S0 = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    nrm, _ = api.orient_samples(bvh, S0)
    S = api.Samples(S0.tri, S0.bary, S0.weight, nrm)
    comp = int(np.bincount(info["face_component"]).argmax())
    cv = v[np.unique(f[info["face_component"] == comp])]
    origin = tuple(float(x) for x in 0.5 * (cv.min(0) + cv.max(0)))
    kw = dict(seed=2, walks_per_sample=64, eps=1e-3, max_steps=1024)
    rec, steps, st = api.run_walks(bvh, S, api.Params(kelvin_origin=origin, exterior_query=1, **kw), True, want_stats=True)
    _, steps3, st3 = api.run_walks(bvh, S, api.Params(kelvin_origin=origin, **kw), True, want_stats=True)
    assert st.n_steps < st3.n_steps
    ids = np.sort(np.random.default_rng(0).choice(400, 40, replace=False))
    orc = Oracle(mesh_geom(v, f))
    orec = orc.run_walks_subset(OracleParams(origin=origin, exterior_query=1, **kw), True, smp["tri"], smp["bary"], smp["weight"],
                                ids, 8, normal=nrm.cpu().numpy())
    slots = (ids[:, None] * 64 + np.arange(8)[None, :]).ravel()
    g = steps.cpu().numpy()[slots]
    assert ((g >= 0) == (orec["steps"] >= 0)).mean() >= 0.97
    assert (g == orec["steps"]).mean() >= 0.9, (g == orec["steps"]).mean()
