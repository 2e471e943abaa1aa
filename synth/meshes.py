"""Seeded synthetic triangle meshes (numpy only; float32 vertices, int32 faces).

All closed primitives are wound so that face normals (v1-v0)x(v2-v0) point
OUT of the solid.  No method arithmetic lives here.
"""
from __future__ import annotations

import numpy as np

__all__ = ["icosphere", "torus", "box", "cylinder", "merge_meshes", "transform",
           "two_spheres_torus_scene", "stress_mesh", "mesh_area"]


def _f32(v):
    return np.ascontiguousarray(v, dtype=np.float32)


def _i32(f):
    return np.ascontiguousarray(f, dtype=np.int32)


def mesh_area(verts, faces):
    """Per-face areas in float64 (used by the sample generators)."""
    v = np.asarray(verts, dtype=np.float64)
    a, b, c = v[faces[:, 0]], v[faces[:, 1]], v[faces[:, 2]]
    return 0.5 * np.linalg.norm(np.cross(b - a, c - a), axis=1)


def icosphere(level: int, radius: float = 1.0, center=(0.0, 0.0, 0.0)):
    """Icosahedron subdivided `level` times, vertices pushed to the sphere.

    V = 10*4^level + 2, F = 20*4^level (level 2: 162 / 320; level 4: 2562 / 5120).
    """
    t = (1.0 + 5.0 ** 0.5) / 2.0
    v = np.array([[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0],
                  [0, -1, t], [0, 1, t], [0, -1, -t], [0, 1, -t],
                  [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array([[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
                  [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
                  [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
                  [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]], dtype=np.int64)
    for _ in range(level):
        nv = v.shape[0]
        e = np.concatenate([f[:, [0, 1]], f[:, [1, 2]], f[:, [2, 0]]], axis=0)
        e_sorted = np.sort(e, axis=1)
        key = e_sorted[:, 0] * nv + e_sorted[:, 1]
        uniq, inv = np.unique(key, return_inverse=True)
        a, b = uniq // nv, uniq % nv
        mid = v[a] + v[b]
        mid /= np.linalg.norm(mid, axis=1, keepdims=True)
        v = np.concatenate([v, mid], axis=0)
        nf = f.shape[0]
        m01, m12, m20 = nv + inv[:nf], nv + inv[nf:2 * nf], nv + inv[2 * nf:]
        f = np.concatenate([
            np.stack([f[:, 0], m01, m20], 1), np.stack([f[:, 1], m12, m01], 1),
            np.stack([f[:, 2], m20, m12], 1), np.stack([m01, m12, m20], 1)], axis=0)
    # make sure of outward winding
    a, b, c = v[f[:, 0]], v[f[:, 1]], v[f[:, 2]]
    flip = np.einsum("ij,ij->i", np.cross(b - a, c - a), a + b + c) < 0
    f[flip] = f[flip][:, [0, 2, 1]]
    v = v * radius + np.asarray(center, dtype=np.float64)
    return _f32(v), _i32(f)


def _grid_faces(nu, nv_, wrap_u, wrap_v, base=0):
    """Two triangles per quad of a (nu x nv_) vertex grid; index = i*nv_ + j."""
    iu = np.arange(nu if wrap_u else nu - 1)
    jv = np.arange(nv_ if wrap_v else nv_ - 1)
    i, j = np.meshgrid(iu, jv, indexing="ij")
    i, j = i.ravel(), j.ravel()
    i1, j1 = (i + 1) % nu, (j + 1) % nv_
    a, b, c, d = i * nv_ + j, i1 * nv_ + j, i1 * nv_ + j1, i * nv_ + j1
    return np.concatenate([np.stack([a, b, c], 1), np.stack([a, c, d], 1)], 0) + base


def torus(R=1.0, r=0.3, n_major=200, n_minor=100, axis="x", center=(0.0, 0.0, 0.0)):
    """Torus with n_major*n_minor quads (2 triangles each), symmetry axis `axis`."""
    u = np.linspace(0.0, 2 * np.pi, n_major, endpoint=False)
    w = np.linspace(0.0, 2 * np.pi, n_minor, endpoint=False)
    uu, ww = np.meshgrid(u, w, indexing="ij")
    x = (R + r * np.cos(ww)) * np.cos(uu)
    y = (R + r * np.cos(ww)) * np.sin(uu)
    z = r * np.sin(ww)
    v = np.stack([x, y, z], -1).reshape(-1, 3)          # axis = z
    f = _grid_faces(n_major, n_minor, True, True)
    if axis == "x":
        v = v[:, [2, 0, 1]]                              # cyclic permutation keeps orientation
    elif axis == "y":
        v = v[:, [1, 2, 0]]
    v, f = _orient_outward_closed(v, f)
    return _f32(v + np.asarray(center)), _i32(f)


def _signed_volume(v, f):
    a, b, c = v[f[:, 0]], v[f[:, 1]], v[f[:, 2]]
    return np.einsum("ij,ij->i", a, np.cross(b, c)).sum() / 6.0


def _orient_outward_closed(v, f):
    if _signed_volume(np.asarray(v, np.float64), f) < 0:
        f = f[:, [0, 2, 1]]
    return v, f


def box(size=(1.0, 1.0, 1.0), segs=(4, 4, 4), center=(0.0, 0.0, 0.0)):
    """Axis-aligned box; each of the 6 faces is its own vertex grid (seams are not welded)."""
    sx, sy, sz = size
    vs, fs, base = [], [], 0
    for ax in range(3):
        a1, a2 = (ax + 1) % 3, (ax + 2) % 3
        n1, n2 = segs[a1] + 1, segs[a2] + 1
        g1 = np.linspace(-0.5, 0.5, n1)
        g2 = np.linspace(-0.5, 0.5, n2)
        p1, p2 = np.meshgrid(g1, g2, indexing="ij")
        for sgn in (-0.5, 0.5):
            v = np.zeros((n1 * n2, 3))
            v[:, ax] = sgn
            v[:, a1] = p1.ravel()
            v[:, a2] = p2.ravel()
            f = _grid_faces(n1, n2, False, False, base)
            if sgn < 0:
                f = f[:, [0, 2, 1]]
            vs.append(v)
            fs.append(f)
            base += n1 * n2
    v = np.concatenate(vs) * np.array([sx, sy, sz])
    f = np.concatenate(fs)
    v, f = _orient_outward_closed(v, f)
    return _f32(v + np.asarray(center)), _i32(f)


def cylinder(radius=0.5, height=1.0, n_theta=64, n_h=4, center=(0.0, 0.0, 0.0)):
    """Capped cylinder about z.  n_h = 1 with large n_theta gives sliver side strips."""
    th = np.linspace(0, 2 * np.pi, n_theta, endpoint=False)
    hz = np.linspace(-0.5 * height, 0.5 * height, n_h + 1)
    tt, hh = np.meshgrid(th, hz, indexing="ij")
    side = np.stack([radius * np.cos(tt), radius * np.sin(tt), hh], -1).reshape(-1, 3)
    f_side = _grid_faces(n_theta, n_h + 1, True, False)
    nb = side.shape[0]
    caps_v = np.array([[0, 0, -0.5 * height], [0, 0, 0.5 * height]])
    i = np.arange(n_theta)
    i1 = (i + 1) % n_theta
    bot = np.stack([np.full(n_theta, nb), i1 * (n_h + 1), i * (n_h + 1)], 1)
    top = np.stack([np.full(n_theta, nb + 1), i * (n_h + 1) + n_h, i1 * (n_h + 1) + n_h], 1)
    v = np.concatenate([side, caps_v])
    f = np.concatenate([f_side, bot, top])
    v, f = _orient_outward_closed(v, f)
    return _f32(v + np.asarray(center)), _i32(f)


def transform(verts, scale=1.0, rotation=None, translation=(0.0, 0.0, 0.0)):
    v = np.asarray(verts, np.float64) * scale
    if rotation is not None:
        v = v @ np.asarray(rotation, np.float64).T
    return _f32(v + np.asarray(translation, np.float64))


def merge_meshes(meshes):
    """Concatenate (verts, faces) pairs into one triangle soup; also returns the
    component id of every vertex and every face."""
    vs, fs, vid, fid, base = [], [], [], [], 0
    for k, (v, f) in enumerate(meshes):
        vs.append(np.asarray(v, np.float32))
        fs.append(np.asarray(f, np.int64) + base)
        vid.append(np.full(len(v), k, np.int32))
        fid.append(np.full(len(f), k, np.int32))
        base += len(v)
    return (_f32(np.concatenate(vs)), _i32(np.concatenate(fs)),
            np.concatenate(vid), np.concatenate(fid))


def two_spheres_torus_scene(level=5, distance=2.5, with_torus=True):
    """BASELINE config 2: two unit icospheres with centres `distance` apart on the
    x axis, plus a torus (R=1, r=0.3, 200x100 quads = 40k triangles) between them
    with its symmetry axis along x."""
    parts = [icosphere(level, 1.0, (-0.5 * distance, 0, 0)),
             icosphere(level, 1.0, (+0.5 * distance, 0, 0))]
    if with_torus:
        parts.append(torus(1.0, 0.3, 200, 100, axis="x"))
    return merge_meshes(parts)


def _random_rotation(rng):
    q = rng.normal(size=4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def _noise_sphere(level, rng, amp):
    v, f = icosphere(level)
    v = v.astype(np.float64)
    disp = np.zeros(len(v))
    for _ in range(6):
        w = rng.normal(size=3) * rng.uniform(1.0, 4.0)
        disp += rng.uniform(0.3, 1.0) * np.sin(v @ w + rng.uniform(0, 2 * np.pi))
    disp *= amp / 6.0
    return _f32(v * (1.0 + disp)[:, None]), f


def _aspect(verts, faces):
    """Longest edge over shortest altitude, L^2 / (2A) (inf for zero area)."""
    v = np.asarray(verts, np.float64)
    a, b, c = v[faces[:, 0]], v[faces[:, 1]], v[faces[:, 2]]
    l2 = np.maximum(np.maximum(((b - a) ** 2).sum(1), ((c - b) ** 2).sum(1)), ((a - c) ** 2).sum(1))
    area = 0.5 * np.linalg.norm(np.cross(b - a, c - a), axis=1)
    with np.errstate(divide="ignore", invalid="ignore"):
        return np.where(area > 0, l2 / (2.0 * area), np.inf)


def stress_mesh(n_faces=2_000_000, n_components=30, seed=3, box_side=6.0,
                sliver_frac=0.05, dup_frac=0.01, flip_frac=0.02):
    """BASELINE config 3 / 4 style 'in-the-wild' mesh: `n_components` overlapping
    and disjoint noise-displaced spheres, boxes and cylinders in a cube of side
    `box_side`; about `sliver_frac` of the faces are slivers with aspect ratio
    > 100 (near-collinear splits plus thin strips on some cylinder sides);
    `dup_frac` of the faces are exact duplicates; `flip_frac` have reversed
    winding.  Returns (verts, faces, info); info holds per-face masks measured on
    the final mesh and the component ids."""
    rng = np.random.default_rng(seed)
    n_dup = int(round(n_faces * dup_frac))
    n_sliver = int(round(n_faces * sliver_frac))
    n_strip_cyl = max(n_components // 10, 1) if n_components >= 3 else 0
    strip_each = (n_sliver // 5) // max(n_strip_cyl, 1) if n_strip_cyl else 0
    n_split = n_sliver - strip_each * n_strip_cyl
    base_target = n_faces - n_dup - 2 * n_split
    n_fill = 1
    n_free = max(n_components - n_strip_cyl - n_fill, 1)
    shares = rng.dirichlet(np.full(n_free, 2.0)) * 0.85 * (base_target - 2 * strip_each * n_strip_cyl)
    kinds = rng.choice(2, size=n_free, p=[0.65, 0.35])
    raw = []
    for k in range(n_free):
        target = max(int(shares[k]), 20)
        if kinds[k] == 0:
            level = int(np.clip(np.floor(np.log(target / 20.0) / np.log(4.0)), 0, 9))
            raw.append(_noise_sphere(level, rng, amp=rng.uniform(0.1, 0.4)))
        else:
            n = max(int(np.sqrt(target / 12.0)), 1)
            raw.append(box(rng.uniform(0.5, 2.0, size=3), (n, n, n)))
    for _ in range(n_strip_cyl):
        n_theta = max(strip_each // 2, 8)          # 2*n_theta thin side triangles
        raw.append(cylinder(rng.uniform(0.2, 0.4), rng.uniform(2.0, 3.0), n_theta, 1))
    used = sum(len(f) for _, f in raw)
    rest = base_target - used                        # fill cylinder with square-ish quads
    if rest >= 16:
        m = max(int(np.sqrt(rest / 2.0 / 3.0)), 2)   # rows of side quads + cap fan
        n_theta = max(rest // (2 * m), 4)
        raw.append(cylinder(0.5, 0.5 * 2 * np.pi * (m - 1) / n_theta if m > 1 else 1.0, n_theta, m - 1))
    parts = []
    for v, f in raw:
        s = rng.uniform(0.3, 1.0)
        tr = rng.uniform(-0.5 * box_side + 1.0, 0.5 * box_side - 1.0, size=3)
        parts.append((transform(v, s, _random_rotation(rng), tr), f))
    verts, faces, vid, fid = merge_meshes(parts)
    faces = faces.astype(np.int64)
    n_split = max(min((n_faces - n_dup - len(faces)) // 2, len(faces)), 0)
    # near-collinear splits: (a,b,c) -> (a,m,c), (m,b,c) and the sliver (a,b,m)
    v64 = verts.astype(np.float64)
    good = np.flatnonzero(_aspect(verts, faces) < 10.0)
    pick = rng.choice(good, size=min(n_split, len(good)), replace=False)
    n_split = len(pick)
    a, b, c = faces[pick, 0], faces[pick, 1], faces[pick, 2]
    mid = 0.5 * (v64[a] + v64[b])
    m = mid + 0.004 * (v64[c] - mid)
    m_idx = len(verts) + np.arange(n_split, dtype=np.int64)
    verts = _f32(np.concatenate([v64, m]))
    vid = np.concatenate([vid, vid[a]])
    faces[pick] = np.stack([a, m_idx, c], 1)
    faces = np.concatenate([faces, np.stack([m_idx, b, c], 1), np.stack([a, b, m_idx], 1)])
    fid = np.concatenate([fid, fid[pick], fid[pick]])
    # duplicated faces (exact copies of existing index triples)
    n_dup = max(n_faces - len(faces), 0)
    dup = rng.choice(len(faces), size=n_dup, replace=False) if n_dup else np.zeros(0, np.int64)
    dup_mask = np.zeros(len(faces) + n_dup, bool)
    dup_mask[len(faces):] = True
    faces = np.concatenate([faces, faces[dup]])
    fid = np.concatenate([fid, fid[dup]])
    # random normal flips
    flip = rng.random(len(faces)) < flip_frac
    faces[flip] = faces[flip][:, [0, 2, 1]]
    faces = _i32(faces)
    info = dict(vertex_component=vid, face_component=fid, sliver=_aspect(verts, faces) > 100.0,
                duplicate=dup_mask, flipped=flip, n_components=len(parts))
    return verts, faces, info
