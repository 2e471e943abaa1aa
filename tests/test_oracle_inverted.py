"""Pins for the oracle's exact distance to Kelvin-inverted faces (reading E4; "inverted triangle
meshes with spherical-triangular elements and ... (non-planar) distance queries"): the closed form (Apollonius sphere
touching the plane / ratio of quadratics on an edge / vertices) against dense sampling of the face IN KELVIN SPACE, i.e.
against the definition min_p |kappa(x) - kappa(p)|; against the conservative radius E3 (which it must dominate, with
equality when all surface points are equally far from the inversion centre); and the exterior walks that use it."""
import numpy as np
import pytest

from oracle import Oracle, OracleParams, inverted_ratio2_triangle, mesh_geom, steklov_eigs
from synth import box, icosphere, vertex_cell_samples


def _kelvin(p):
    return p / (p ** 2).sum(-1, keepdims=True)


def _grid_bary(n):
    i, j = np.meshgrid(np.arange(n + 1), np.arange(n + 1), indexing="ij")
    keep = i + j <= n
    u, v = i[keep] / n, j[keep] / n
    return np.stack([1 - u - v, u, v], 1)


def test_inverted_triangle_distance_is_the_minimum_over_the_inverted_face():
    """d(y, kappa(T)) = sqrt(ratio2) / |x| must equal min over a dense sample of T of |y - kappa(p)|, where y = kappa(x):
    never above any sampled value, and within the sampling resolution of the smallest one; the reported barycentrics
    reproduce the value."""
    rng = np.random.default_rng(0)
    B = _grid_bary(240)
    n_face = n_edge = n_vertex = 0
    for trial in range(300):
        a, b, c = rng.normal(size=(3, 3)) * rng.uniform(0.2, 2.0) + rng.normal(size=3) * rng.uniform(0.0, 2.0)
        if trial % 7 == 0:
            c = a + (b - a) * rng.uniform(0.2, 0.8) + 1e-3 * rng.normal(size=3)          # sliver
        x = rng.normal(size=3) * rng.uniform(0.3, 3.0)
        if trial % 3 == 0:                                                                # x over the face: interior minimiser
            w = rng.dirichlet([2, 2, 2])
            nrm = np.cross(b - a, c - a)
            x = w @ np.stack([a, b, c]) + nrm / np.linalg.norm(nrm) * rng.normal() * 0.3
        if min(np.linalg.norm(a), np.linalg.norm(b), np.linalg.norm(c)) < 0.05:
            continue
        r2, bary = inverted_ratio2_triangle(x, a, b, c)
        assert (bary >= -1e-12).all() and abs(bary.sum() - 1) < 1e-12
        p = bary @ np.stack([a, b, c])
        assert abs(((x - p) ** 2).sum() / (p ** 2).sum() - r2) <= 1e-12 * max(r2, 1.0)    # the minimiser gives the value
        P = B @ np.stack([a, b, c])
        y = _kelvin(x)
        d_samples = np.linalg.norm(y - _kelvin(P), axis=1)                               # the definition, in Kelvin space
        d_closed = np.sqrt(r2) / np.linalg.norm(x)
        assert d_closed <= d_samples.min() * (1 + 1e-12) + 1e-15
        # resolution of the sample: neighbouring grid points of the inverted face are at most this far apart
        L = max(np.linalg.norm(a - b), np.linalg.norm(b - c), np.linalg.norm(c - a))
        res = 2.0 * L / 240 / np.linalg.norm(P, axis=1).min() ** 2
        assert d_samples.min() - d_closed <= res, (trial, d_samples.min(), d_closed, res)
        nz = (bary > 1e-9).sum()
        n_face += nz == 3; n_edge += nz == 2; n_vertex += nz == 1
    assert n_face > 40 and n_edge > 40 and n_vertex > 20                                 # all three branches are exercised


def test_inverted_distance_special_cases():
    # x on the face: distance 0.  x at a vertex: 0.
    a, b, c = np.array([1.0, 0, 0.5]), np.array([0, 1.0, 0.5]), np.array([-1.0, -1.0, 0.5])
    r2, bary = inverted_ratio2_triangle(0.2 * a + 0.3 * b + 0.5 * c, a, b, c)
    assert r2 < 1e-24
    assert inverted_ratio2_triangle(b, a, b, c)[0] == 0.0
    # plane z = h = 0.5, huge face, x on the axis at height t: the inverted plane is the sphere of diameter 1/h = 2 through 0
    # (centre (0, 0, 1)), and y = kappa(x) = (0, 0, 1/t) lies on its axis.  The nearest point of that sphere is its top
    # pole (0, 0, 2) = kappa of the foot (0, 0, h) while y is above the centre (t < 1): distance |1/t - 1/h|; below the
    # centre (t > 1) it is the bottom pole 0 = kappa(infinity), which the finite face only approaches: distance -> 1/t.
    big = 1e4
    A, B_, C_ = np.array([big, 0, 0.5]), np.array([-big, big, 0.5]), np.array([-big, -big, 0.5])
    for t in (0.1, 0.3, 0.8):
        r2, bary = inverted_ratio2_triangle(np.array([0, 0, t]), A, B_, C_)
        assert abs(np.sqrt(r2) / t - abs(1 / t - 1 / 0.5)) < 1e-9
        assert np.abs(bary @ np.stack([A, B_, C_]) - [0, 0, 0.5]).max() < 1e-6
    for t in (2.0, 7.0):
        r2, bary = inverted_ratio2_triangle(np.array([0, 0, t]), A, B_, C_)
        assert abs(np.sqrt(r2) / t - 1 / t) < 1e-3 / t and np.linalg.norm(bary @ np.stack([A, B_, C_])) > 0.5 * big
    # x -> infinity: kappa(x) -> 0, and the nearest point of the inverted face is the image of the face point FARTHEST
    # from the inversion centre: ratio -> |x| / max |p|
    xf = np.array([1e9, 2e9, -1e9])
    r2, bary = inverted_ratio2_triangle(xf, a, b, c)
    far = max(np.linalg.norm(a), np.linalg.norm(b), np.linalg.norm(c))
    assert abs(np.sqrt(r2) * far / np.linalg.norm(xf) - 1.0) < 1e-6 and abs(np.linalg.norm(bary @ np.stack([a, b, c])) - far) < 1e-6


def test_exact_inverted_radius_dominates_the_conservative_one():
    """Reading E3's radius D / (rho min(R_max, rho + D)) is a lower bound of the exact distance to the inverted surface
    (SURVEY.md 8(c)); on a sphere about the inversion centre every |p| is equal and the two agree (up to the faceting)."""
    rng = np.random.default_rng(1)
    v, f = box((1.0, 2.0, 0.7), (3, 3, 3))
    orc = Oracle(mesh_geom(v, f))
    o = np.array([0.1, -0.2, 0.05])
    Rmax = orc.max_vertex_norm(o)
    ratios = []
    for _ in range(200):
        x = o + rng.normal(size=3) * rng.uniform(0.8, 4.0)
        r = orc.closest_points(x[None].astype(np.float32))
        x32 = x.astype(np.float32).astype(np.float64)
        if np.all(np.abs(x32 - o) < np.array([0.5, 1.0, 0.35]) * 0.98):                    # inside the box: not exterior
            continue
        D, rho = r["dist"][0], np.linalg.norm(x32 - o)
        e3 = D / (rho * min(Rmax, rho + D))
        ratio, tri, cp, bary = orc.closest_point_inverted(x32, o)
        exact = ratio / rho
        assert exact >= e3 * (1 - 1e-7), (exact, e3)
        ratios.append(e3 / exact)
    assert len(ratios) > 100 and min(ratios) < 0.9 and np.mean(ratios) > 0.5             # a real bound, and not a wild one
    v, f = icosphere(4)
    orc = Oracle(mesh_geom(v, f))
    for _ in range(50):
        x = rng.normal(size=3); x *= rng.uniform(1.05, 5.0) / np.linalg.norm(x)
        x32 = x.astype(np.float32).astype(np.float64)
        D, rho = orc.closest_points(x32[None].astype(np.float32))["dist"][0], np.linalg.norm(x32)
        ratio, tri, cp, bary = orc.closest_point_inverted(x32, (0, 0, 0))
        assert abs(ratio / rho - D / (rho * min(1.0, rho + D))) < 2e-3 * (ratio / rho) + 1e-4


def test_exterior_walks_with_the_exact_inverted_query():
    """Same estimator, larger balls: the walks with E4 take fewer jumps than with E3, end on the surface, and give the
    exterior sphere spectrum l + 1 (with the killing term) like the E3 walks do."""
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 4, seed=0)
    orc = Oracle(mesh_geom(v, f))
    M = orc.mass_matrix()
    origin = (0.25, 0.1, -0.15)
    out = {}
    for q in (0, 1):
        P = OracleParams(seed=4, walks_per_sample=96, eps=1e-3, include_killing=True, n_kill_walks=40_000, origin=origin,
                         exterior_query=q)
        res = orc.estimate_dtn(P, True, smp["tri"], smp["bary"], smp["weight"], want_var=True)
        rec = res["records"]
        assert (rec["steps"] >= 0).all()
        t = rec["t"]
        assert np.abs(np.linalg.norm(t, axis=1) - 1.0).max() < 0.02                        # exit points on the (faceted) sphere
        out[q] = (res["S"], res["var"], rec["steps"].mean(), steklov_eigs(res["S"], M, 9))
    assert out[1][2] < 0.9 * out[0][2], (out[0][2], out[1][2])                             # fewer jumps
    lam = out[1][3]
    assert abs(lam[0] - 1.0) < 0.08 and abs(lam[1:4].mean() - 2.0) < 0.2 and abs(lam[4:9].mean() - 3.0) < 0.35
    # the two variants estimate the same matrix
    err = np.linalg.norm(out[0][0] - out[1][0])
    se = np.sqrt(np.linalg.norm(np.sqrt(out[0][1])) ** 2 + np.linalg.norm(np.sqrt(out[1][1])) ** 2)
    assert err < 1.5 * se, (err, se)
