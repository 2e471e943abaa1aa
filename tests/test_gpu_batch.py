"""mcs_estimate_dtn_batch (BASELINE config 4: many meshes, dense K x K operators per mesh): every mesh's matrices are
bit-identical to the single calls (build -> sidedness -> mcs_estimate_dtn_both), whatever the number of workers."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from synth import fps_samples, icosphere, stress_mesh, vertex_cell_samples     # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


def _stress_item(api, seed, n_faces, n_comp, K=128):
    v, f, info = stress_mesh(n_faces=n_faces, n_components=n_comp, seed=seed)
    smp = fps_samples(v, f, K, n_candidates=6000, seed=seed)
    comp = int(np.bincount(info["face_component"]).argmax())
    cv = v[np.unique(f[info["face_component"] == comp])]
    origin = tuple(float(x) for x in 0.5 * (cv.min(0) + cv.max(0)))
    a, b, c = v[f[smp["tri"], 0]], v[f[smp["tri"], 1]], v[f[smp["tri"], 2]]
    pts = (smp["bary"][:, 0:1] * a + smp["bary"][:, 1:2] * b + smp["bary"][:, 2:3] * c).astype(np.float32)
    return dict(verts=torch.as_tensor(v).cuda(), faces=torch.as_tensor(f).cuda(),
                samples=api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"]), origin=origin,
                pts=torch.as_tensor(pts).cuda())


def test_batch_equals_the_single_calls_bit_for_bit(api):
    items = [_stress_item(api, s, nf, nc) for s, nf, nc in ((0, 6000, 3), (1, 20000, 9), (2, 9000, 1), (3, 40000, 20), (4, 5000, 2))]
    Pi = api.Params(seed=7, walks_per_sample=128, eps=1e-3)
    Pe = api.Params(seed=7, walks_per_sample=128, eps=1e-3, far_alpha=0.5, far_near_factor=4.0)
    K = 128
    # single calls: the reference
    ref = []
    for m in items:
        bvh = api.build_bvh(m["verts"], m["faces"])
        nrm, _ = api.orient_samples_fast(bvh, m["samples"], beta=2.5)
        S = api.Samples(m["samples"].tri, m["samples"].bary, m["samples"].weight, nrm)
        basis = api.PointBasis(m["pts"], nrm, k=8, sigma=0.025, tau_n=0.8)
        import dataclasses
        a, b = api.estimate_dtn_both(bvh, S, Pi, dataclasses.replace(Pe, kelvin_origin=m["origin"]), basis=basis)
        ref.append((a.clone(), b.clone(), nrm.clone()))
    for workers in (1, 3):
        oi = torch.full((len(items), K, K), float("nan"), device="cuda")
        oe = torch.full((len(items), K, K), float("nan"), device="cuda")
        # the point basis uses the sidedness normals, which the batch call computes itself: two passes, as a caller
        # without precomputed normals would do (first the normals, then the bases)
        batch = [dict(m) for m in items]
        for m, r in zip(batch, ref):
            m["basis"] = api.PointBasis(m["pts"], r[2], k=8, sigma=0.025, tau_n=0.8)
        normals = api.estimate_dtn_batch(batch, Pi, Pe, oi, oe, orient_h_scale=1.0, orient_beta=2.5, n_workers=workers)
        for i, r in enumerate(ref):
            assert torch.equal(normals[i], r[2])
            assert torch.equal(oi[i], r[0]) and torch.equal(oe[i], r[1]), (workers, i)


def test_batch_hat_basis_and_error_reporting(api):
    meshes = []
    for level in (1, 2, 2):
        v, f = icosphere(level)
        smp = vertex_cell_samples(v, f, 2, seed=level)
        meshes.append(dict(verts=torch.as_tensor(v).cuda(), faces=torch.as_tensor(f).cuda(),
                           samples=api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"]), origin=(0.1, 0.0, 0.0)))
    Pi = api.Params(seed=1, walks_per_sample=64, eps=1e-3)
    Pe = api.Params(seed=1, walks_per_sample=64, eps=1e-3, include_killing=True, n_kill_walks=3000)
    oi = [torch.empty((m["verts"].shape[0],) * 2, device="cuda") for m in meshes]
    oe = [torch.empty((m["verts"].shape[0],) * 2, device="cuda") for m in meshes]
    api.estimate_dtn_batch(meshes, Pi, Pe, oi, oe, orient_h_scale=0.0, n_workers=2)
    import dataclasses
    for m, a, b in zip(meshes, oi, oe):
        bvh = api.build_bvh(m["verts"], m["faces"])
        ra, rb = api.estimate_dtn_both(bvh, m["samples"], Pi, dataclasses.replace(Pe, kelvin_origin=m["origin"]))
        assert torch.equal(a, ra) and torch.equal(b, rb)
    # a broken mesh in the middle: its code is reported, the others are still computed
    bad = dict(meshes[1]); bad["faces"] = bad["faces"].clone(); bad["faces"][0, 0] = 10_000
    oi2 = [torch.zeros_like(x) for x in oi]; oe2 = [torch.zeros_like(x) for x in oe]
    with pytest.raises(api.McsError) as e:
        api.estimate_dtn_batch([meshes[0], bad, meshes[2]], Pi, Pe, oi2, oe2, orient_h_scale=0.0, n_workers=2)
    assert e.value.code == api.MCS_EINVAL and "(1," in str(e.value)
    assert torch.equal(oi2[0], oi[0]) and torch.equal(oe2[2], oe[2])
