"""Seeded closest-point query sets ('Tie-free query set').
Only the raw candidates are generated here; the tie filter needs distances and
therefore lives in the tests, where it calls the oracle."""
from __future__ import annotations

import numpy as np

__all__ = ["near_surface_queries", "far_field_queries"]


def near_surface_queries(verts, faces, n: int, seed: int = 0):
    """Interior point of a random triangle (barycentrics >= 0.15) displaced along
    the face normal by h in [1e-3, 0.3] * local edge length, random side."""
    rng = np.random.default_rng(seed)
    v = np.asarray(verts, np.float64)
    f = np.asarray(faces, np.int64)[rng.integers(len(faces), size=n)]
    b = rng.dirichlet(np.ones(3), size=n) * 0.55 + 0.15
    a, bb, c = v[f[:, 0]], v[f[:, 1]], v[f[:, 2]]
    p = b[:, 0:1] * a + b[:, 1:2] * bb + b[:, 2:3] * c
    nrm = np.cross(bb - a, c - a)
    ln = np.linalg.norm(nrm, axis=1, keepdims=True)
    ok = ln[:, 0] > 0
    nrm = np.where(ln > 0, nrm / np.maximum(ln, 1e-300), 0.0)
    edge = np.linalg.norm(bb - a, axis=1)
    h = np.exp(rng.uniform(np.log(1e-3), np.log(0.3), size=n)) * edge
    side = np.where(rng.random(n) < 0.5, -1.0, 1.0)
    q = p + (side * h)[:, None] * nrm
    return np.ascontiguousarray(q[ok], np.float32)


def far_field_queries(verts, n: int, seed: int = 0, scale: float = 3.0):
    """Uniform points in the mesh AABB scaled by `scale` about its centre."""
    rng = np.random.default_rng(seed)
    v = np.asarray(verts, np.float64)
    lo, hi = v.min(0), v.max(0)
    c, h = 0.5 * (lo + hi), 0.5 * (hi - lo) * scale
    return np.ascontiguousarray(c + (rng.random((n, 3)) * 2 - 1) * h, np.float32)
