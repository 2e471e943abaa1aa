"""Pins for the oracle's point-based k-NN bilateral basis (Eq. 44-45):
neighbour search against numpy, special cases of the weights, partition of unity, and the closed-form sphere
spectrum through the whole estimator (no GPU)."""
import numpy as np
import pytest

from oracle import Oracle, OracleParams, PointBasis, mesh_geom, sphere_geom
from sph import DEGREES, fibonacci_sphere, real_sph_harm


def test_knn_indices_match_numpy_stable_argsort():
    rng = np.random.default_rng(0)
    pts = rng.normal(size=(300, 3)).astype(np.float32)
    pts[50] = pts[10]                                         # an exact tie: the smaller index must come first
    nrm = pts / np.linalg.norm(pts, axis=1, keepdims=True)
    pb = PointBasis(pts, nrm, k=8, sigma=0.5, tau_n=0.8)
    q = np.concatenate([rng.normal(size=(40, 3)), pts[[10]].astype(np.float64)])
    idx, w = Oracle(sphere_geom()).knn_weights(pb, q, np.tile([0.0, 0.0, 1.0], (len(q), 1)))
    d2 = ((q[:, None, :] - pts[None].astype(np.float64)) ** 2).sum(2)
    want = np.argsort(d2, axis=1, kind="stable")[:, :8]
    assert np.array_equal(idx, want)
    assert idx[-1, 0] == 10 and idx[-1, 1] == 50
    assert np.allclose(w.sum(1), 1.0, atol=1e-14) and (w >= 0).all()


def test_weight_special_cases():
    orc = Oracle(sphere_geom())
    # two points at equal distance: only the normals decide, ratio exp((c1 - c2) / tau)
    pts = np.array([[1, 0, 0], [-1, 0, 0]], np.float32)
    nrm = np.array([[0, 0, 1], [0, 1, 0]], np.float32)
    pb = PointBasis(pts, nrm, k=2, sigma=0.7, tau_n=0.8)
    idx, w = orc.knn_weights(pb, [[0, 0, 0]], [[0, 0, 1]])
    assert idx.tolist() == [[0, 1]] and abs(w[0, 0] / w[0, 1] - np.exp(1 / 0.8)) < 1e-12
    # equal normals: only the distances decide, ratio exp((d2^2 - d1^2) / (2 sigma^2))
    pb = PointBasis(pts, np.tile([0, 0, 1], (2, 1)).astype(np.float32), k=2, sigma=0.7, tau_n=0.8)
    idx, w = orc.knn_weights(pb, [[0.5, 0, 0]], [[0, 0, 1]])
    assert idx.tolist() == [[0, 1]] and abs(w[0, 0] / w[0, 1] - np.exp((1.5 ** 2 - 0.5 ** 2) / (2 * 0.49))) < 1e-9
    # k = 1: the indicator of the nearest point;  sigma, tau -> infinity: uniform 1/k
    rng = np.random.default_rng(1)
    pts = rng.normal(size=(64, 3)).astype(np.float32)
    nrm = pts / np.linalg.norm(pts, axis=1, keepdims=True)
    q = rng.normal(size=(20, 3))
    idx, w = orc.knn_weights(PointBasis(pts, nrm, k=1), q, q)
    assert (w == 1.0).all() and np.array_equal(idx[:, 0], ((q[:, None] - pts[None]) ** 2).sum(2).argmin(1))
    idx, w = orc.knn_weights(PointBasis(pts, nrm, k=8, sigma=1e6, tau_n=1e9), q, q)
    assert np.abs(w - 0.125).max() < 1e-9
    # [Rk1] many sigma away from every point: still a partition of unity (no 0/0), dominated by the nearest
    idx, w = orc.knn_weights(PointBasis(pts, nrm, k=8, sigma=1e-3, tau_n=0.8), q * 50, q)
    assert np.isfinite(w).all() and np.allclose(w.sum(1), 1.0) and (w[:, 0] > 0.999).all()
    # [Rk3] k larger than the number of points
    idx, w = orc.knn_weights(PointBasis(pts[:3], nrm[:3], k=8, sigma=1.0), q[:2], q[:2])
    assert (idx[:, 3:] == -1).all() and np.allclose(w[:, :3].sum(1), 1.0) and (w[:, 3:] == 0).all()


def test_point_basis_sphere_spectrum_closed_form():
    """Unit ball, K quasi-uniform points with radial normals: for g = Y_l sampled at the points,
    g^T S g / g^T M g (lumped mass 4 pi / K) must be l (cap 0.5 deg: minus about (l + 1) sin(theta0 / 2)) when the
    interpolator is sharp (sigma = 0.35 point spacings), and LOWER when it smooths (sigma = one spacing);
    constants are annihilated exactly (partition of unity); S is symmetric PSD."""
    K, n_s, W = 600, 6000, 32
    pts = fibonacci_sphere(K)
    spacing = float(np.sqrt(4 * np.pi / K))
    pos = fibonacci_sphere(n_s)
    orc = Oracle(sphere_geom((0, 0, 0), 1.0))
    P = OracleParams(seed=5, walks_per_sample=W, eps=1e-5, rmax=0.5 * 1024 / 1023, cap_half_angle_deg=0.5)
    wgt = np.full(n_s, 4 * np.pi / n_s, np.float32)
    rec, _ = orc.run_walks(P, False, weight=wgt, pos=pos)
    Y = real_sph_harm(pts)                                    # [K, n_modes], orthonormal on the sphere
    lams = {}
    for fac in (0.35, 1.0):
        pb = PointBasis(pts, pts, k=8, sigma=fac * spacing, tau_n=0.8)
        S = orc.accumulate_points(pb, rec, weight=wgt, pos=pos)
        assert np.abs(S - S.T).max() < 1e-12 * np.abs(S).max()
        assert np.abs(S.sum(1)).max() < 1e-10 * np.abs(S).max()
        assert np.linalg.eigvalsh(S).min() > -1e-10 * np.abs(S).max()
        lams[fac] = np.array([Y[:, j] @ S @ Y[:, j] / (4 * np.pi / K * (Y[:, j] @ Y[:, j])) for j in range(Y.shape[1])])
    for j, l in enumerate(DEGREES):
        assert abs(lams[0.35][j] - l) < 0.05 * l + 0.03, (l, lams[0.35][j])
    j4 = list(DEGREES).index(4)
    assert lams[1.0][j4] < lams[0.35][j4] - 0.3               # a wide kernel smooths the high degrees


def test_point_basis_on_mesh_equals_hat_basis_in_the_limit_k1_points_at_exit():
    """k = 1 with the points = the mesh vertices: b(q) is the indicator of the nearest vertex.  The matrix is then a
    coarser quadrature of the same operator: symmetric PSD, zero row sums, same trace order as the hat basis."""
    from synth import icosphere, vertex_cell_samples
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 2, seed=0)
    orc = Oracle(mesh_geom(v, f))
    nrm = v / np.linalg.norm(v, axis=1, keepdims=True)
    P = OracleParams(seed=1, walks_per_sample=32, eps=1e-3)
    out = orc.estimate_dtn_points(PointBasis(v, nrm, k=1), P, False, smp["tri"], smp["bary"], smp["weight"])
    S = out["S"]
    assert np.abs(S - S.T).max() < 1e-14 and np.abs(S.sum(1)).max() < 1e-12
    assert np.linalg.eigvalsh(S).min() > -1e-12
    Sh = orc.accumulate_hat(out["records"], smp["tri"], smp["bary"])
    assert 0.5 < np.trace(S) / np.trace(Sh) < 10.0           # indicator functions jump by 1 where hats change by less
