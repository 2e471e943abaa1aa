"""The whole pipeline on a handful of seeded in-the-wild style meshes (BASELINE config 4 in small: slivers,
duplicates, flipped faces, 1-30 components): build, winding-number sidedness, interior and exterior (killing on)
in the k-NN point basis and in the hat basis (sparse output), eigenpairs.  No oracle here -- the properties that
hold for any input: no error, finite, exactly symmetric, PSD to rounding, interior constants in the kernel,
bit-identical reruns, every walk accounted for.  (A mesh of this kind once broke the exterior walk kernel.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from synth import fps_samples, stress_mesh                                     # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


@pytest.mark.parametrize("seed", range(8))
def test_pipeline_properties(api, seed):
    rng = np.random.default_rng(1000 + seed)
    n_faces = int(np.exp(rng.uniform(np.log(3e3), np.log(6e4))))
    v, f, info = stress_mesh(n_faces=n_faces, n_components=int(rng.integers(1, 31)), seed=500 + seed)
    n_s, W = 256, int(rng.choice([16, 64, 256]))
    smp = fps_samples(v, f, n_s, n_candidates=6000, seed=seed)
    bvh = api.build_bvh(torch.from_numpy(v).cuda(), torch.from_numpy(f).cuda())
    S0 = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    nrm, d = api.orient_samples(bvh, S0)
    assert torch.isfinite(nrm).all() and torch.isfinite(d).all()
    S = api.Samples(S0.tri, S0.bary, S0.weight, nrm)
    comp = np.bincount(info["face_component"]).argmax()
    cv = v[np.unique(f[info["face_component"] == comp])]
    origin = tuple(float(x) for x in 0.5 * (cv.min(0) + cv.max(0)))
    tv = v[f[smp["tri"]]].astype(np.float64)
    pts = np.einsum("qk,qkd->qd", smp["bary"].astype(np.float64), tv).astype(np.float32)
    pb = api.PointBasis(torch.from_numpy(pts).cuda(), nrm, k=8, sigma=0.15, tau_n=0.8)
    Pi = api.Params(seed=seed, walks_per_sample=W, eps=1e-3, max_steps=256)
    Pe = api.Params(seed=seed, walks_per_sample=W, eps=1e-3, max_steps=256, include_killing=True, n_kill_walks=4096,
                    kelvin_origin=origin)
    mats = []
    for ext, P in ((False, Pi), (True, Pe)):
        fn = api.estimate_dtn_exterior if ext else api.estimate_dtn_interior
        A, st = fn(bvh, S, P, basis=pb, want_stats=True)
        assert torch.equal(A, fn(bvh, S, P, basis=pb))
        assert torch.isfinite(A).all() and torch.equal(A, A.T)
        assert st.n_walks == n_s * W + (4096 if ext else 0)
        rec, steps = api.run_walks(bvh, S, P, ext)
        steps = steps.cpu().numpy()
        assert st.n_truncated == int(((steps == -1) | (steps == -3)).sum())
        assert (steps >= 0).mean() > 0.5
        An = A.double().cpu().numpy()
        assert np.linalg.eigvalsh(An).min() > -1e-4 * np.abs(An).max()
        if not ext:
            assert np.abs(An.sum(1)).max() < 2e-4 * np.abs(An).max()
        coo = api.estimate_dtn_coo(bvh, S, P, exterior=ext)
        assert coo.nnz > 0 and torch.isfinite(coo.val).all()
        assert bool((coo.row <= coo.col).all())
        mats.append(A)
    mass = torch.from_numpy(smp["weight"].astype(np.float32)).cuda()
    lam, psi, sweeps = api.steklov_eigs(torch.stack(mats), torch.stack([mass, mass]), 32)
    assert sweeps < 30 and torch.isfinite(lam).all() and torch.isfinite(psi).all()
    assert bool((lam[:, 1:] >= lam[:, :-1]).all())
    scale = (mats[0].diag() / mass).max().item()                                 # an upper bound of the spectrum's order of magnitude
    assert abs(lam[0, 0].item()) < 1e-4 * scale                                  # interior: the constant mode
