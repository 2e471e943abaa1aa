"""GPU parity of mcs_steklov_eigs against the oracle's LAPACK step:
eigenvalues to fp32 accuracy of the matrix scale, eigenvectors M-orthonormal with small residuals and -- where the
eigenvalue is isolated -- equal to the oracle's up to sign; multiplets are compared as subspaces."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import Oracle, OracleParams, mesh_geom, steklov_eigpairs          # noqa: E402
from synth import icosphere, vertex_cell_samples                               # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


def _check(S, m, lam, psi, n_eig):
    """Compare one GPU result with the oracle."""
    S = np.asarray(S, np.float64); m = np.asarray(m, np.float64)
    w, V = steklov_eigpairs(S, m, n_eig)
    Ssym = 0.5 * (S + S.T)
    scale = np.abs(np.linalg.eigvalsh(Ssym / np.sqrt(np.outer(m, m)))).max()
    assert np.abs(lam - w).max() < 2e-5 * scale
    assert np.all(np.diff(lam) >= 0)
    if psi is None:
        return
    assert np.abs((psi * m) @ psi.T - np.eye(n_eig)).max() < 5e-5                      # M-orthonormal
    res = Ssym @ psi.T - (m[:, None] * psi.T) * lam[None, :]
    assert np.abs(res / np.sqrt(m)[:, None]).max() < 5e-5 * scale                      # residual in the M^-1/2 scaling
    gap = np.minimum(np.diff(w, prepend=-np.inf), np.diff(w, append=np.inf))           # needs all K to be exact at the top
    for e in range(n_eig - 1):
        if gap[e] > 1e-2 * scale:                                                       # isolated: the vector is unique up to sign
            c = (psi[e] * m) @ V[e]
            assert abs(abs(c) - 1) < 1e-4
    # every GPU vector lies in the span of oracle vectors with nearby eigenvalues
    wa, Va = steklov_eigpairs(S, m, len(S))
    for e in range(n_eig):
        near = np.abs(wa - lam[e]) < 1e-2 * scale
        c = (Va[near] * m) @ psi[e]
        assert abs(np.linalg.norm(c) - 1) < 2e-3


@pytest.mark.parametrize("K,n_eig", [(1, 1), (2, 2), (5, 3), (17, 17), (64, 10), (130, 9), (257, 20), (385, 8), (512, 64), (600, 16), (700, 5), (896, 6), (901, 12), (1800, 8)])
def test_random_spd_pencils(api, K, n_eig):
    rng = np.random.default_rng(K)
    A = rng.normal(size=(K, K + 3))
    S = (A @ A.T / K).astype(np.float32)
    m = rng.uniform(0.3, 2.0, K).astype(np.float32)
    lam, psi, sweeps = api.steklov_eigs(torch.from_numpy(S).cuda(), torch.from_numpy(m).cuda(), n_eig, method="jacobi")
    assert 1 <= sweeps < 30 or K == 1
    _check(S, m, lam.cpu().numpy().astype(np.float64), psi.cpu().numpy().astype(np.float64), n_eig)
    lam2, none, _ = api.steklov_eigs(torch.from_numpy(S).cuda(), torch.from_numpy(m).cuda(), n_eig, want_vectors=False, method="jacobi")
    assert none is None and torch.equal(lam, lam2)                                     # values do not depend on the vector output


def test_large_matrix_takes_the_row_pair_path(api):
    """K > 3520: the rows no longer fit in shared memory; row pairs are rotated in place (DtN-like spectrum)."""
    K, n_eig = 3600, 6
    rng = np.random.default_rng(1)
    Q, _ = np.linalg.qr(rng.normal(size=(K, K)))
    S = ((Q * (2.0 * np.sqrt(np.arange(K)))) @ Q.T).astype(np.float32)
    m = np.ones(K, np.float32)
    lam, psi, sweeps = api.steklov_eigs(torch.from_numpy(S).cuda(), torch.from_numpy(m).cuda(), n_eig, method="jacobi")
    assert sweeps < 30
    _check(S, m, lam.cpu().numpy().astype(np.float64), psi.cpu().numpy().astype(np.float64), n_eig)


def test_batch_equals_single_and_is_deterministic(api):
    rng = np.random.default_rng(7)
    B, K, n_eig = 5, 96, 12
    A = rng.normal(size=(B, K, K))
    S = np.einsum("bij,bkj->bik", A, A).astype(np.float32) / K
    m = rng.uniform(0.5, 1.5, (B, K)).astype(np.float32)
    Sg, mg = torch.from_numpy(S).cuda(), torch.from_numpy(m).cuda()
    lam, psi, _ = api.steklov_eigs(Sg, mg, n_eig)
    lam_b, psi_b, _ = api.steklov_eigs(Sg, mg, n_eig)
    assert torch.equal(lam, lam_b) and torch.equal(psi, psi_b)
    for b in range(B):
        _check(S[b], m[b], lam[b].cpu().numpy().astype(np.float64), psi[b].cpu().numpy().astype(np.float64), n_eig)
    # a matrix solved alone converges on its own schedule: same eigenpairs to solver accuracy
    l0, p0, _ = api.steklov_eigs(Sg[2], mg[2], n_eig)
    assert (l0 - lam[2]).abs().max().item() < 1e-5 * lam[2].abs().max().item() + 1e-6


def test_singular_and_multiplet_spectrum(api):
    """Cycle Laplacian: a null vector (constants) and double eigenvalues 2 - 2 cos(2 pi j / n) -- the structure of
    an interior DtN matrix (constants in the kernel)."""
    n = 90
    S = (2 * np.eye(n) - np.roll(np.eye(n), 1, 0) - np.roll(np.eye(n), -1, 0)).astype(np.float32)
    m = np.full(n, 0.5, np.float32)
    lam, psi, _ = api.steklov_eigs(torch.from_numpy(S).cuda(), torch.from_numpy(m).cuda(), 11)
    lam, psi = lam.cpu().numpy().astype(np.float64), psi.cpu().numpy().astype(np.float64)
    expect = np.sort(2 * (2 - 2 * np.cos(2 * np.pi * np.arange(n) / n)))[:11]
    assert np.abs(lam - expect).max() < 2e-5 * 8
    assert np.abs(np.abs(psi[0]) - np.sqrt(2.0 / n)).max() < 1e-4
    _check(S, m, lam, psi, 11)


def test_spectrum_of_an_estimated_dtn_matrix(api):
    """The end of the pipeline: eigenpairs of the GPU-estimated interior DtN matrix of the unit sphere, against the
    oracle's LAPACK on the same matrix, and the first multiplets near the closed form l = 0, 1, 2."""
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 4, seed=0)
    bvh = api.build_bvh(torch.from_numpy(v).cuda(), torch.from_numpy(f).cuda())
    S = api.estimate_dtn_interior(bvh, api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"]),
                                  api.Params(seed=5, walks_per_sample=128, eps=1e-3))
    tv = v[f].astype(np.float64)
    area = 0.5 * np.linalg.norm(np.cross(tv[:, 1] - tv[:, 0], tv[:, 2] - tv[:, 0]), axis=1)
    mass = np.bincount(f.ravel(), weights=np.repeat(area / 3.0, 3), minlength=len(v))       # lumped mass: vertex cell areas
    mg = torch.from_numpy(mass.astype(np.float32)).cuda()
    lam, psi, _ = api.steklov_eigs(S, mg, 9)
    _check(S.cpu().numpy(), mass.astype(np.float32), lam.cpu().numpy().astype(np.float64), psi.cpu().numpy().astype(np.float64), 9)
    lam = lam.cpu().numpy()
    assert abs(lam[0]) < 0.05 and np.all(np.abs(lam[1:4] - 1) < 0.25) and np.all(np.abs(lam[4:9] - 2) < 0.5)


def _check_subspace(S, m, lam, psi, n_eig, tol_rel=1e-4):
    """Subspace iteration stops on residuals (2e-5 of the Gershgorin bound), so its bars are set from the matrix scale:
    eigenvalues to tol_rel * scale (second order in the residual), vectors as subspaces of near eigenvalues."""
    S = np.asarray(S, np.float64); m = np.asarray(m, np.float64)
    wa, Va = steklov_eigpairs(S, m, len(S))
    scale = np.abs(wa).max()
    assert np.abs(lam - wa[:n_eig]).max() < tol_rel * scale
    assert np.all(np.diff(lam) >= 0)
    assert np.abs((psi * m) @ psi.T - np.eye(n_eig)).max() < 5e-5                      # M-orthonormal
    Ssym = 0.5 * (S + S.T)
    res = Ssym @ psi.T - (m[:, None] * psi.T) * lam[None, :]
    assert np.abs(np.linalg.norm(res / np.sqrt(m)[:, None], axis=0)).max() < 1e-3 * scale
    for e in range(n_eig):
        near = np.abs(wa - lam[e]) < 2e-2 * scale
        c = (Va[near] * m) @ psi[e]
        assert abs(np.linalg.norm(c) - 1) < 2e-3


@pytest.mark.parametrize("K,n_eig,kind", [(1024, 16, "sqrt"), (1500, 64, "sqrt"), (2562, 40, "sphere"), (1300, 100, "sqrt")])
def test_subspace_iteration_for_few_eigenpairs_of_a_large_matrix(api, K, n_eig, kind):
    """DtN-like spectra: lambda_n ~ sqrt(n) (a surface: eigenvalue l has multiplicity ~ 2l + 1), or exactly the sphere's
    l with multiplicity 2l + 1 -- whole multiplets inside and across the end of the block."""
    rng = np.random.default_rng(K + n_eig)
    Q, _ = np.linalg.qr(rng.normal(size=(K, K)))
    if kind == "sqrt":
        w = np.sqrt(np.arange(K))
    else:
        w = np.floor(np.sqrt(np.arange(K))).astype(np.float64)                          # 0, 1 x3, 2 x5, 3 x7, ...
    S = ((Q * w) @ Q.T).astype(np.float32)
    m = rng.uniform(0.5, 2.0, K).astype(np.float32)
    Sg, mg = torch.from_numpy(S).cuda(), torch.from_numpy(m).cuda()
    lam, psi, iters = api.steklov_eigs(Sg, mg, n_eig, method="subspace")
    assert 1 <= iters <= 40
    _check_subspace(S, m, lam.cpu().numpy().astype(np.float64), psi.cpu().numpy().astype(np.float64), n_eig)
    # deterministic, the automatic choice takes the same path, and the values do not depend on the vector output
    lam2, psi2, _ = api.steklov_eigs(Sg, mg, n_eig)
    assert torch.equal(lam, lam2) and torch.equal(psi, psi2)
    lam3, none, _ = api.steklov_eigs(Sg, mg, n_eig, want_vectors=False, method="subspace")
    assert none is None and torch.equal(lam, lam3)
    # against the Jacobi solver of the same library
    lam_j, _, _ = api.steklov_eigs(Sg, mg, n_eig, method="jacobi", want_vectors=False)
    assert (lam - lam_j).abs().max().item() < 1e-4 * float(np.abs(w).max())


def test_subspace_iteration_batch_and_fallback(api):
    rng = np.random.default_rng(3)
    K, n_eig, B = 1100, 20, 2
    S = np.empty((B, K, K), np.float32); m = rng.uniform(0.5, 2.0, (B, K)).astype(np.float32)
    for b in range(B):
        Q, _ = np.linalg.qr(rng.normal(size=(K, K)))
        S[b] = ((Q * np.sqrt((b + 1.0) * np.arange(K))) @ Q.T).astype(np.float32)
    lam, psi, _ = api.steklov_eigs(torch.from_numpy(S).cuda(), torch.from_numpy(m).cuda(), n_eig, method="subspace")
    for b in range(B):
        _check_subspace(S[b], m[b], lam[b].cpu().numpy().astype(np.float64), psi[b].cpu().numpy().astype(np.float64), n_eig)
    # where subspace iteration does not apply it is refused; the automatic choice takes Jacobi there
    with pytest.raises(api.McsError):
        api.steklov_eigs(torch.eye(512, device="cuda"), torch.ones(512, device="cuda"), 8, method="subspace")
    with pytest.raises(api.McsError):
        api.steklov_eigs(torch.from_numpy(S[0]).cuda(), torch.from_numpy(m[0]).cuda(), 600, method="subspace")
    # a spectrum crowded at its low end (Wishart): whatever the filter achieves, the automatic choice returns converged pairs
    A = rng.normal(size=(K, K + 3))
    W = (A @ A.T / K).astype(np.float32)
    lam_a, psi_a, _ = api.steklov_eigs(torch.from_numpy(W).cuda(), torch.from_numpy(m[0]).cuda(), 8)
    _check(W, m[0], lam_a.cpu().numpy().astype(np.float64), psi_a.cpu().numpy().astype(np.float64), 8)


def test_argument_errors(api):
    S = torch.eye(4, device="cuda"); m = torch.ones(4, device="cuda")
    with pytest.raises(api.McsError):
        api.steklov_eigs(S, m, 5)
    with pytest.raises(api.McsError):
        api.steklov_eigs(S, m, 0)
