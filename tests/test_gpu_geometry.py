"""GPU parity, geometry half (SURVEY.md 8(c) "LBVH (GPU)", "Tie-free query set"):
Philox words, the radix sort, LBVH invariants, and closest-point queries against the
brute-force fp64 oracle -- face index bit-exact on tie-free queries, distance within
1e-6 relative.  Everything goes through the C ABI (paper_2606_05581_b200.api)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import Oracle, mesh_geom, philox4x32_10 as orc_philox          # noqa: E402
from synth import (box, cylinder, far_field_queries, icosphere, merge_meshes,    # noqa: E402
                   near_surface_queries, stress_mesh, torus, two_spheres_torus_scene)


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


def _cuda(a, dtype):
    return torch.as_tensor(np.ascontiguousarray(a)).to(device="cuda", dtype=dtype)


def _bvh(api, v, f):
    return api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))


# ------------------------------------------------------------------------------
def test_philox_words_match_oracle_bit_exact(api):
    rng = np.random.default_rng(0)
    ctr = rng.integers(0, 2 ** 32, size=(4096, 4), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0
    ctr[1] = 0xFFFFFFFF
    key = (0x9E3779B9, 0x12345678)
    out = api.philox4x32_10(_cuda(ctr.view(np.int32), torch.int32), key).cpu().numpy().view(np.uint32)
    for i in list(range(64)) + [4095]:
        assert tuple(int(x) for x in out[i]) == orc_philox(ctr[i], key)


@pytest.mark.parametrize("n,bits", [(0, 64), (1, 64), (1000, 64), (300_001, 63), (70_000, 17)])
def test_radix_sort_is_stable_and_exact(api, n, bits):
    rng = np.random.default_rng(n + bits)
    hi = (1 << min(bits, 62))
    keys = rng.integers(0, hi, size=n, dtype=np.int64)
    if n > 100:
        keys[: n // 2] = keys[n // 2: n // 2 * 2] if n % 2 == 0 else keys[n // 2 + 1:]   # many duplicates
    vals = np.arange(n, dtype=np.int32)
    k, v = api.sort_pairs_u64(_cuda(keys, torch.int64), _cuda(vals, torch.int32), bits)
    order = np.argsort(keys, kind="stable")
    assert np.array_equal(k.cpu().numpy(), keys[order])
    assert np.array_equal(v.cpu().numpy(), vals[order])


def _unpack_nodes(nodes):
    w = nodes.cpu().numpy()
    f = w.view(np.float32)
    box0 = f[:, 0:6]
    box1 = f[:, 6:12]
    return box0, box1, w[:, 12], w[:, 13], w[:, 14]


MESHES = {
    "icosphere3": lambda: icosphere(3),
    "torus": lambda: torus(1.0, 0.3, 60, 30),
    "scene": lambda: two_spheres_torus_scene(level=3, distance=2.5, with_torus=True)[:2],
    "stress20k": lambda: stress_mesh(n_faces=20_000, n_components=8, seed=3)[:2],
}


@pytest.mark.parametrize("split", [False, True])
@pytest.mark.parametrize("name", list(MESHES))
def test_lbvh_invariants(api, name, split):
    """Structure of the packed tree.  split=False: one leaf per face.  split=True (the default build): long thin
    faces enter as several leaf references, one per slab across their longest edge; every face
    keeps at least one leaf, an unsplit face has exactly its vertex box, and the slab boxes of a split face cover it."""
    v, f = MESHES[name]()
    F = len(f)
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32), split=split)
    info = bvh.info()
    R = info.n_leaves
    assert info.F == F and info.n_nodes == R - 1 and info.V == len(v)
    assert R == F if not split else F <= R <= 2 * F                   # default budget: one extra leaf per face on average
    nodes, leaf_tri, morton = bvh.dump()
    box0, box1, c0, c1, parent = _unpack_nodes(nodes)
    m = morton.cpu().numpy().astype(np.uint64)
    assert len(m) == R and (m[1:] >= m[:-1]).all()                    # keys sorted
    lt = leaf_tri.cpu().numpy()
    per_face = np.bincount(lt, minlength=F)
    assert len(lt) == R and per_face.min() >= 1 and per_face.sum() == R   # every face in at least one leaf
    if not split:
        assert per_face.max() == 1
    children = np.concatenate([c0, c1])
    leaves = ~children[children < 0]
    inner = children[children >= 0]
    assert np.array_equal(np.sort(leaves), np.arange(R))              # every leaf reference hangs in the tree once
    assert np.array_equal(np.sort(inner), np.arange(1, R - 1))        # every node but the root has one parent
    assert parent[0] == -1
    leaf_box = np.zeros((R, 6), np.float32)
    for c, boxes in ((c0, box0), (c1, box1)):
        isleaf = c < 0
        leaf_box[~c[isleaf]] = boxes[isleaf]
        # child box = union of the grandchildren's boxes, and parent links agree
        ii = c[~isleaf]
        lo = np.minimum(box0[ii][:, :3], box1[ii][:, :3])
        hi = np.maximum(box0[ii][:, 3:], box1[ii][:, 3:])
        assert np.array_equal(boxes[~isleaf][:, :3], lo) and np.array_equal(boxes[~isleaf][:, 3:], hi)
        assert np.array_equal(parent[ii], np.nonzero(~isleaf)[0])
    # an unsplit face lies in its leaf box exactly (the box is the min/max of its fp32 vertices)
    single = per_face[lt] == 1
    tv = v[f[lt[single]]]
    assert np.array_equal(leaf_box[single][:, :3], tv.min(1)) and np.array_equal(leaf_box[single][:, 3:], tv.max(1))
    # a split face: long and thin, and every point of it lies in at least one of its slab boxes
    multi = np.flatnonzero(per_face > 1)
    if split and name == "stress20k":
        assert len(multi) > 50
    if len(multi):
        vv = v.astype(np.float64)
        a, b, c = vv[f[multi, 0]], vv[f[multi, 1]], vv[f[multi, 2]]
        L2 = np.maximum(np.maximum(((b - a) ** 2).sum(1), ((c - b) ** 2).sum(1)), ((a - c) ** 2).sum(1))
        area2 = np.linalg.norm(np.cross(b - a, c - a), axis=1)
        assert (L2 > 7.9 * area2).all()                               # aspect L^2 / 2A > 8
        rng = np.random.default_rng(0)
        w = rng.dirichlet(np.ones(3), size=64)                        # random interior points ...
        w = np.concatenate([w, np.eye(3), [[0.5, 0.5, 0], [0, 0.5, 0.5], [0.5, 0, 0.5]],     # ... corners, edge midpoints,
                            np.stack([np.linspace(0, 1, 33), 1 - np.linspace(0, 1, 33), np.zeros(33)], 1),   # and the edges
                            np.stack([np.zeros(33), np.linspace(0, 1, 33), 1 - np.linspace(0, 1, 33)], 1),
                            np.stack([1 - np.linspace(0, 1, 33), np.zeros(33), np.linspace(0, 1, 33)], 1)])
        order = np.argsort(lt, kind="stable")
        start = np.concatenate([[0], np.cumsum(per_face)])
        for k, face in enumerate(multi[:400]):
            pts = w @ np.stack([a[k], b[k], c[k]])
            bx = leaf_box[order[start[face]:start[face + 1]]].astype(np.float64)
            inside = ((pts[:, None, :] >= bx[None, :, :3]) & (pts[:, None, :] <= bx[None, :, 3:])).all(2).any(1)
            assert inside.all(), (face, per_face[face])
            tvf = v[f[face]]
            assert (bx[:, :3].min(0) <= tvf.min(0)).all() and (bx[:, 3:].max(0) >= tvf.max(0)).all()
    # area and AABB against numpy on the same fp32 inputs
    vv = v.astype(np.float64)
    area = 0.5 * np.linalg.norm(np.cross(vv[f[:, 1]] - vv[f[:, 0]], vv[f[:, 2]] - vv[f[:, 0]]), axis=1).sum()
    assert abs(info.area - area) <= 1e-9 * area
    used = np.unique(f)
    assert np.array_equal(np.array(info.aabb_lo[:]), v[used].min(0)) and np.array_equal(np.array(info.aabb_hi[:]), v[used].max(0))
    assert info.max_depth >= int(np.ceil(np.log2(F)))
    assert info.sah_cost > 0.0


def test_sliver_splitting_lowers_the_tree_cost_and_changes_no_query(api):
    """Stress mesh with rotated sliver strips: the surface-area cost of the tree drops with the default build, the
    closest-point results are bit-identical with and without splitting (every reference carries the whole triangle),
    and so are the walk records of both operators."""
    v, f, info = stress_mesh(n_faces=60_000, n_components=12, seed=5)
    vd, fd = _cuda(v, torch.float32), _cuda(f, torch.int32)
    b0, b1 = api.build_bvh(vd, fd, split=False), api.build_bvh(vd, fd)
    i0, i1 = b0.info(), b1.info()
    assert i1.n_leaves > i0.n_leaves == len(f)
    assert i1.sah_cost < 0.7 * i0.sah_cost, (i0.sah_cost, i1.sah_cost)
    q = np.concatenate([near_surface_queries(v, f, 30000, seed=5), far_field_queries(v, 10000, seed=6)])
    qd = _cuda(q, torch.float32)
    r0, r1 = api.closest_point(b0, qd), api.closest_point(b1, qd)
    assert all(torch.equal(x, y) for x, y in zip(r0, r1))
    from synth import fps_samples
    smp = fps_samples(v, f, 256, n_candidates=10_000, seed=1)
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    comp = int(np.bincount(info["face_component"]).argmax())
    cv = v[np.unique(f[info["face_component"] == comp])]
    origin = tuple(float(x) for x in 0.5 * (cv.min(0) + cv.max(0)))
    for ext in (False, True):
        P = api.Params(seed=2, walks_per_sample=128, eps=1e-3, kelvin_origin=origin)
        ra, sa, sta = api.run_walks(b0, S, P, ext, want_stats=True)
        rb, sb, stb = api.run_walks(b1, S, P, ext, want_stats=True)
        assert torch.equal(ra.view(torch.int32), rb.view(torch.int32)) and torch.equal(sa, sb)
        assert stb.n_tris_tested < sta.n_tris_tested               # fewer triangle tests for the same walks


def _tie_free(orc, q, rel_gap=1e-4):
    """SURVEY.md 8(c) tie filter, decided by the oracle in fp64: keep a query when every
    other face (exact copies of the winner aside: those are resolved by the index rule)
    is farther than the winner by more than rel_gap * best."""
    r = orc.closest_points(q)
    keep = (orc.runner_up(q, r["tri"]) - r["dist"]) > rel_gap * r["dist"]
    return keep, r


def _copy_classes(f):
    """Class id per face: faces with the same three vertices (any order) share a class.
    `reordered[c]` is True when a class holds copies with DIFFERENT vertex order: their
    distances agree only up to rounding, so they are near-ties, not exact ties."""
    key = np.sort(f.astype(np.int64), axis=1)
    _, cls = np.unique(key, axis=0, return_inverse=True)
    cls = cls.ravel()
    first = np.full(cls.max() + 1, -1, np.int64)
    first[cls[::-1]] = np.arange(len(f))[::-1]
    reordered = np.zeros(cls.max() + 1, bool)
    diff = (f != f[first[cls]]).any(1)
    reordered[cls[diff]] = True
    return cls, reordered


@pytest.mark.parametrize("name", list(MESHES))
def test_closest_point_matches_oracle_on_tie_free_queries(api, name):
    v, f = MESHES[name]()
    orc = Oracle(mesh_geom(v, f))
    q = np.concatenate([near_surface_queries(v, f, 6000, seed=1), far_field_queries(v, 3000, seed=2)])
    keep, r = _tie_free(orc, q)
    cls, reordered = _copy_classes(f)
    keep &= ~reordered[cls[r["tri"]]]
    assert keep.sum() > 2000
    bvh = _bvh(api, v, f)
    dist, tri, bary = api.closest_point(bvh, _cuda(q, torch.float32))
    dist, tri, bary = dist.cpu().numpy(), tri.cpu().numpy(), bary.cpu().numpy()
    assert np.array_equal(tri[keep], r["tri"][keep])                  # bit-exact face index
    scale = float(np.abs(v).max())
    D = r["dist"]
    big = D >= 1e-2 * scale
    assert (np.abs(dist - D)[keep & big] <= 1e-6 * D[keep & big]).all()
    assert (np.abs(dist - D)[keep & ~big] <= 2e-7 * scale).all()
    # all queries (ties included): distance still agrees; barycentrics reproduce the closest point
    assert (np.abs(dist - D) <= 1e-6 * D + 2e-7 * scale).all()
    cp = np.einsum("qk,qkd->qd", bary.astype(np.float64), v[f[tri]].astype(np.float64))
    assert (np.abs(np.linalg.norm(cp - q, axis=1) - D) <= 2e-6 * D + 4e-7 * scale).all()
    assert (bary >= 0).all() and np.abs(bary.sum(1) - 1).max() < 1e-6


@pytest.mark.parametrize("name", ["scene", "stress20k"])
def test_bvh_query_equals_device_bruteforce_bitwise(api, name):
    """Same fp32 point-triangle routine, same tie rule => the tree must not change a bit."""
    v, f = MESHES[name]()
    bvh = _bvh(api, v, f)
    q = np.concatenate([near_surface_queries(v, f, 20000, seed=5), far_field_queries(v, 10000, seed=6),
                        v[f[:500, 0]], (v[f[:500, 0]] + v[f[:500, 1]]) / 2])       # exact ties: vertices, edge midpoints
    qd = _cuda(q, torch.float32)
    d1, t1, b1 = api.closest_point(bvh, qd)
    d2, t2, b2 = api.closest_point_bruteforce(bvh, qd)
    assert torch.equal(d1, d2)
    t1, t2 = t1.cpu().numpy(), t2.cpu().numpy()
    cls, reordered = _copy_classes(f)
    exact = ~reordered[cls[t2]]
    assert np.array_equal(t1[exact], t2[exact])                  # exact ties included: smaller index wins
    assert np.array_equal(cls[t1], cls[t2])                      # reordered copies: the same triangle
    assert torch.equal(b1[torch.as_tensor(exact, device="cuda")], b2[torch.as_tensor(exact, device="cuda")])


def test_duplicate_and_degenerate_faces(api):
    """Duplicated faces tie exactly -> smaller index wins; zero-area faces absorb as segments."""
    v, f = icosphere(2)
    f2 = np.concatenate([f, f[:40]])                                   # duplicates with larger indices
    v2 = np.concatenate([v, np.array([[2, 0, 0], [3, 0, 0], [2.5, 0, 0]], np.float32)])
    f2 = np.concatenate([f2, np.array([[len(v), len(v) + 1, len(v) + 2]], np.int32)])   # collinear face
    bvh = _bvh(api, v2, f2)
    assert bvh.info().n_degenerate == 1
    cen = v[f[:40]].mean(1) * 1.05
    q = np.concatenate([cen, np.array([[2.25, 0.5, 0.0], [4.0, 0, 0]], np.float32)])
    dist, tri, _ = api.closest_point(bvh, _cuda(q, torch.float32))
    tri, dist = tri.cpu().numpy(), dist.cpu().numpy()
    assert np.array_equal(tri[:40], np.arange(40))
    assert tri[40] == len(f2) - 1 and abs(dist[40] - 0.5) < 1e-6
    assert tri[41] == len(f2) - 1 and abs(dist[41] - 1.0) < 1e-6


def test_build_edge_cases_and_errors(api):
    v = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0]], np.float32)
    f = np.array([[0, 1, 2]], np.int32)
    bvh = _bvh(api, v, f)                                              # single face
    d, t, b = api.closest_point(bvh, _cuda(np.array([[0.25, 0.25, 2.0], [2, 0, 0]]), torch.float32))
    assert t.tolist() == [0, 0] and abs(d[0].item() - 2.0) < 1e-6 and abs(d[1].item() - 1.0) < 1e-6
    d, t, b = api.closest_point(bvh, torch.empty((0, 3), device="cuda"))       # empty query set
    assert d.numel() == 0
    with pytest.raises(api.McsError) as e:
        _bvh(api, v, np.array([[0, 1, 3]], np.int32))                   # index out of range
    assert e.value.code == api.MCS_EINVAL
    with pytest.raises(api.McsError) as e:
        _bvh(api, np.array([[0, 0, 0], [1, 0, 0], [np.nan, 1, 0]], np.float32), f)
    assert e.value.code == api.MCS_EDEGENERATE
    with pytest.raises(api.McsError) as e:
        _bvh(api, np.array([[0, 0, 0], [1, 0, 0], [2, 0, 0]], np.float32), f)   # zero total area
    assert e.value.code == api.MCS_EDEGENERATE
    # two faces
    v2, f2 = np.concatenate([v, [[1, 1, 0]]]).astype(np.float32), np.array([[0, 1, 2], [1, 3, 2]], np.int32)
    bvh = _bvh(api, v2, f2)
    d, t, _ = api.closest_point(bvh, _cuda(np.array([[0.9, 0.9, 1.0]]), torch.float32))
    assert t.item() == 1 and abs(d.item() - 1.0) < 1e-6


def test_closest_point_one_million_queries(api):
    """SURVEY.md 8(c) 'LBVH (GPU)': query result = brute force on >= 1e6 queries.  The exhaustive device scan
    (same fp32 point-triangle routine, every face) is the brute force at this count; the fp64 oracle checks a
    seeded sample of them, tie-free by its own gap filter."""
    v, f = two_spheres_torus_scene(level=4, distance=2.5, with_torus=True)[:2]
    q = np.concatenate([near_surface_queries(v, f, 700_000, seed=21), far_field_queries(v, 300_000, seed=22)])
    bvh = _bvh(api, v, f)
    qd = _cuda(q, torch.float32)
    d1, t1, b1 = api.closest_point(bvh, qd)
    d2, t2, b2 = api.closest_point_bruteforce(bvh, qd)
    assert torch.equal(d1, d2) and torch.equal(t1, t2) and torch.equal(b1, b2)
    idx = np.random.default_rng(3).choice(len(q), 4000, replace=False)
    orc = Oracle(mesh_geom(v, f))
    keep, r = _tie_free(orc, q[idx])
    assert keep.sum() > 1500                                       # symmetric scene: many far-field queries are near-ties
    assert np.array_equal(t1.cpu().numpy()[idx][keep], r["tri"][keep])
    D, dg = r["dist"], d1.cpu().numpy()[idx]
    assert (np.abs(dg - D) <= 1e-6 * D + 2e-7 * float(np.abs(v).max())).all()
