"""Pins for the oracle's closest-point code (no GPU): a second formulation,
geometric invariants, brute force on tiny inputs, and the textbook closed form
of the distance to an axis-aligned box."""
import numpy as np

from oracle import (Oracle, closest_point_triangle, closest_point_triangle_alt, mesh_geom)
from synth import box, icosphere


def _random_triangles(rng, n):
    tris = rng.normal(size=(n, 3, 3))
    # a share of thin slivers and of exactly degenerate (collinear / repeated) faces
    k = n // 4
    tris[:k, 2] = tris[:k, 0] + (tris[:k, 1] - tris[:k, 0]) * rng.uniform(0.1, 0.9, (k, 1)) \
        + 1e-3 * rng.normal(size=(k, 3))
    m = n // 10
    tris[k:k + m, 2] = tris[k:k + m, 0] + 0.25 * (tris[k:k + m, 1] - tris[k:k + m, 0])
    tris[k + m:k + m + 5, 1] = tris[k + m:k + m + 5, 0]
    return tris


def test_region_method_matches_second_formulation_and_invariants():
    rng = np.random.default_rng(1)
    tris = _random_triangles(rng, 400)
    for t in tris:
        a, b, c = t
        for p in rng.normal(size=(12, 3)) * 2.0:
            d2, cp, bary = closest_point_triangle(p, a, b, c)
            d2b, cpb = closest_point_triangle_alt(p, a, b, c)
            scale = 1.0 + np.abs(t).max() ** 2 + p @ p
            assert abs(d2 - d2b) <= 1e-9 * scale
            # invariants: valid barycentrics reproduce the point, which is no farther than any vertex
            assert bary.min() >= -1e-12 and abs(bary.sum() - 1.0) <= 1e-12
            assert np.allclose(bary @ t, cp, atol=1e-9 * np.sqrt(scale))
            assert abs((p - cp) @ (p - cp) - d2) <= 1e-9 * scale
            assert d2 <= min(((p - v) ** 2).sum() for v in t) + 1e-12 * scale


def test_triangle_brute_force_on_barycentric_grid():
    rng = np.random.default_rng(2)
    n = 60
    i, j = np.meshgrid(np.arange(n + 1), np.arange(n + 1), indexing="ij")
    keep = i + j <= n
    w = np.stack([i[keep], j[keep], n - i[keep] - j[keep]], 1) / n
    for _ in range(60):
        t = rng.normal(size=(3, 3))
        p = rng.normal(size=3) * 1.5
        d2, cp, bary = closest_point_triangle(p, *t)
        pts = w @ t
        brute = ((pts - p) ** 2).sum(1).min()
        h = max(np.linalg.norm(t[0] - t[1]), np.linalg.norm(t[1] - t[2]), np.linalg.norm(t[2] - t[0])) / n
        assert d2 <= brute + 1e-12                      # never worse than any sampled point
        assert np.sqrt(brute) <= np.sqrt(d2) + h        # and the grid gets within one cell of it


def _box_distance(p, half):
    """Textbook distance from a point to the SURFACE of the box [-half, half]."""
    q = np.abs(p) - half
    outside = np.linalg.norm(np.maximum(q, 0.0), axis=-1)
    inside = -np.max(q, axis=-1)
    return np.where((q <= 0).all(-1), inside, outside)


def test_mesh_brute_force_equals_box_closed_form():
    size = np.array([1.0, 0.6, 1.4])
    v, f = box(size, (3, 2, 4))
    orc = Oracle(mesh_geom(v, f))
    rng = np.random.default_rng(3)
    q = (rng.random((3000, 3)) * 2 - 1).astype(np.float32) * 1.5
    out = orc.closest_points(q)
    want = _box_distance(q.astype(np.float64), 0.5 * size)
    assert np.abs(out["dist"] - want).max() < 1e-6
    # the closest point lies on the reported face with the reported barycentrics
    tri = f[out["tri"]]
    cp = np.einsum("qk,qkd->qd", out["bary"], v[tri].astype(np.float64))
    assert np.abs(cp - out["cp"]).max() < 1e-12
    assert np.abs(np.linalg.norm(q - out["cp"], axis=1) - out["dist"]).max() < 1e-12


def test_tie_break_prefers_smaller_index():
    v, f = icosphere(1)
    f2 = np.concatenate([f, f[:10]])                     # duplicated faces: exact ties
    orc = Oracle(mesh_geom(v, f2))
    c = v[f[:10]].mean(1) * 1.3
    out = orc.closest_points(c.astype(np.float32))
    assert (out["tri"] == np.arange(10)).all()
    # a vertex is shared by 5-6 faces: the smallest face index among them wins
    out = orc.closest_points((v[:12] * 2).astype(np.float32))
    for k in range(12):
        assert out["tri"][k] == np.flatnonzero((f2 == k).any(1)).min()


def test_sphere_mesh_distance_bounds():
    """A polyhedron inscribed in the unit sphere lies between the spheres of radius
    1 - sag and 1, which brackets the distance from any point on a ray."""
    v, f = icosphere(3)
    orc = Oracle(mesh_geom(v, f))
    rng = np.random.default_rng(4)
    q = rng.normal(size=(500, 3))
    q = (q / np.linalg.norm(q, axis=1, keepdims=True) * rng.uniform(0.2, 2.5, (500, 1))).astype(np.float32)
    out = orc.closest_points(q, want_second=True)
    rho = np.linalg.norm(q.astype(np.float64), axis=1)
    tv = v[f].astype(np.float64)
    nrm = np.cross(tv[:, 1] - tv[:, 0], tv[:, 2] - tv[:, 0])
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    sag = 1.0 - np.einsum("ij,ij->i", nrm, tv[:, 0]).min()      # deepest face plane
    outside = rho >= 1
    inside = rho <= 1 - sag
    assert outside.sum() > 100 and inside.sum() > 100
    assert (out["dist"][outside] >= rho[outside] - 1 - 1e-6).all()
    assert (out["dist"][outside] <= rho[outside] - 1 + sag + 1e-6).all()
    assert (out["dist"][inside] <= 1 - rho[inside] + 1e-6).all()
    assert (out["dist"][inside] >= 1 - sag - rho[inside] - 1e-6).all()
    assert (out["second"] >= out["dist"]).all()
