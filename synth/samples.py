"""Seeded boundary-sample generators: surface points (tri, bary) with quadrature
weights a_i that sum to the surface area.  These are INPUTS of the estimator
(PAPER.md:269 `UniformSampleMesh`; SURVEY.md section 8(c) reading R1); numpy's
PCG64 draws them, not the method's Philox streams.
"""
from __future__ import annotations

import numpy as np

from .meshes import mesh_area

__all__ = ["vertex_cell_samples", "uniform_samples", "fps_samples"]


def _pack(tri, bary, weight, **extra):
    out = dict(tri=np.ascontiguousarray(tri, np.int32),
               bary=np.ascontiguousarray(bary, np.float32),
               weight=np.ascontiguousarray(weight, np.float32))
    out.update(extra)
    return out


def _uniform_in_triangle(rng, n):
    r1 = np.sqrt(rng.random(n))
    r2 = rng.random(n)
    return np.stack([1.0 - r1, r1 * (1.0 - r2), r1 * r2], 1)


def vertex_cell_samples(verts, faces, per_vertex: int, seed: int = 0):
    """`per_vertex` sample points per mesh vertex, drawn uniformly from the
    vertex's barycentric-dual cell (in each incident triangle the quad
    {vertex, two edge midpoints, centroid}); weight = A_cell / per_vertex with
    A_cell = (1/3) * sum of incident triangle areas.  The cells tile the mesh,
    so the weights sum to the total area (stratified version of PAPER.md:269).
    Sample points are never placed at a vertex."""
    rng = np.random.default_rng(seed)
    faces = np.asarray(faces, np.int64)
    nv = len(verts)
    area = mesh_area(verts, faces)
    corner_v = faces.ravel()                      # corner id = 3*f + k
    corner_a = np.repeat(area / 3.0, 3)
    order = np.argsort(corner_v, kind="stable")
    cv, ca = corner_v[order], corner_a[order]
    cum = np.cumsum(ca)
    cell = np.bincount(corner_v, weights=corner_a, minlength=nv)
    start = np.concatenate([[0.0], cum])[np.searchsorted(cv, np.arange(nv), side="left")]
    vert = np.repeat(np.arange(nv), per_vertex)
    vert = vert[cell[vert] > 0]
    u = rng.random(len(vert))
    target = start[vert] + u * cell[vert]
    idx = np.searchsorted(cum, target, side="right")
    idx = np.clip(idx, np.searchsorted(cv, vert, side="left"),
                  np.searchsorted(cv, vert, side="right") - 1)
    corner = order[idx]
    f, k = corner // 3, corner % 3
    # uniform point in the quad (v, m1, centroid, m2), local barycentrics (l_k, l_k+1, l_k+2)
    p0 = np.array([1.0, 0.0, 0.0])
    m1 = np.array([0.5, 0.5, 0.0])
    cen = np.array([1 / 3, 1 / 3, 1 / 3])
    m2 = np.array([0.5, 0.0, 0.5])
    w = _uniform_in_triangle(rng, len(vert))
    first = rng.random(len(vert)) < 0.5
    q1 = np.where(first[:, None], m1, cen)
    q2 = np.where(first[:, None], cen, m2)
    loc = w[:, :1] * p0 + w[:, 1:2] * q1 + w[:, 2:3] * q2
    bary = np.empty_like(loc)
    rows = np.arange(len(vert))
    for j in range(3):
        bary[rows, (k + j) % 3] = loc[:, j]
    weight = cell[vert] / per_vertex
    return _pack(f, bary, weight, vertex=vert.astype(np.int32))


def uniform_samples(verts, faces, n: int, seed: int = 0):
    """n points uniform on the surface, weight = area / n (Eq. 26)."""
    rng = np.random.default_rng(seed)
    area = mesh_area(verts, faces)
    cum = np.cumsum(area)
    tri = np.searchsorted(cum, rng.random(n) * cum[-1], side="right")
    tri = np.minimum(tri, len(faces) - 1)
    bary = _uniform_in_triangle(rng, n)
    return _pack(tri, bary, np.full(n, cum[-1] / n))


_fps_lib = None


def _fps_indices(pts, first: int, n: int):
    """Indices picked by greedy farthest-point sampling (synth/fps.c: bucketed exact search, the same picks
    as the plain numpy loop it replaces, which took minutes on 1 M candidates)."""
    global _fps_lib
    import ctypes as C
    if _fps_lib is None:
        from .build import build
        _fps_lib = C.CDLL(build())
        _fps_lib.synth_fps.restype = C.c_int
    pts = np.ascontiguousarray(pts, np.float32)
    # candidates in Z-order (10 bits per axis) so that fps.c's buckets of consecutive points are compact
    lo, ext = pts.min(0), np.maximum(pts.max(0) - pts.min(0), 1e-30)
    q = np.minimum(((pts - lo) / ext * 1024.0).astype(np.int64), 1023)
    key = np.zeros(len(pts), np.int64)
    for bit in range(10):
        for d in range(3):
            key |= ((q[:, d] >> bit) & 1) << (3 * bit + 2 - d)
    perm = np.argsort(key, kind="stable").astype(np.int64)
    sorted_pts = np.ascontiguousarray(pts[perm])
    first_pos = int(np.flatnonzero(perm == int(first))[0])
    chosen = np.empty(n, np.int64)
    rc = _fps_lib.synth_fps(sorted_pts.ctypes.data_as(C.c_void_p), perm.ctypes.data_as(C.c_void_p), C.c_int64(len(pts)),
                            C.c_int64(first_pos), C.c_int64(n), chosen.ctypes.data_as(C.c_void_p))
    if rc != 0:
        raise ValueError("synth_fps: bad arguments")
    return chosen


def fps_samples(verts, faces, n: int, n_candidates: int = 200_000, seed: int = 0):
    """Greedy farthest-point sampling of n points among `n_candidates`
    area-uniform candidates (BASELINE configs 3-4); weight = area / n."""
    cand = uniform_samples(verts, faces, n_candidates, seed)
    v = np.asarray(verts, np.float64)
    f = np.asarray(faces, np.int64)[cand["tri"]]
    b = cand["bary"].astype(np.float64)
    pts = (b[:, 0:1] * v[f[:, 0]] + b[:, 1:2] * v[f[:, 1]] + b[:, 2:3] * v[f[:, 2]]).astype(np.float32)
    rng = np.random.default_rng(seed + 1)
    chosen = _fps_indices(pts, int(rng.integers(n_candidates)), n)
    total = float(mesh_area(verts, faces).sum())
    return _pack(cand["tri"][chosen], cand["bary"][chosen], np.full(n, total / n))
