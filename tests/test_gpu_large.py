"""BASELINE config 3 at its full face count (2M faces, 30 overlapping / disjoint components, 5 %
slivers, 1 % duplicated faces, 2 % flipped faces): the LBVH build and the queries at the size
where the tree no longer fits in L2, checked against the brute-force oracle on sampled queries and
walks, and against the on-device exhaustive scan.  The matrix itself needs the sparse output for
K = V ~ 1M; records are what is compared here."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import Oracle, OracleParams, mesh_geom                            # noqa: E402
from synth import far_field_queries, fps_samples, near_surface_queries, stress_mesh   # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


@pytest.fixture(scope="module")
def big(api):
    v, f, info = stress_mesh(n_faces=2_000_000, n_components=30, seed=3)
    bvh = api.build_bvh(torch.as_tensor(v).cuda(), torch.as_tensor(f).cuda())
    return v, f, info, bvh, Oracle(mesh_geom(v, f))


def test_build_2m_faces(api, big):
    v, f, info, bvh, orc = big
    bi = bvh.info()
    assert bi.F == 2_000_000 and bi.n_nodes == bi.n_leaves - 1 and bi.F < bi.n_leaves <= 2 * bi.F
    assert 21 <= bi.max_depth <= 96                                   # log2(2M) = 20.9; traversal stack bound
    area = orc.total_area()
    assert abs(bi.area - area) <= 1e-9 * area
    nodes, leaf_tri, morton = bvh.dump()
    m = morton.cpu().numpy().astype(np.uint64)
    assert (m[1:] >= m[:-1]).all()
    lt = leaf_tri.cpu().numpy()
    per_face = np.bincount(lt, minlength=bi.F)
    assert per_face.min() >= 1 and per_face.sum() == bi.n_leaves     # every face has a leaf; long slivers have several
    assert info["sliver"][per_face > 1].all()                         # only slivers were cut (aspect > 100 among them all)
    # tree quality readout: the rotated strips dominate the surface-area cost of the unsplit tree
    plain = api.build_bvh(torch.as_tensor(v).cuda(), torch.as_tensor(f).cuda(), split=False).info()
    assert plain.n_leaves == bi.F and bi.sah_cost < 0.2 * plain.sah_cost, (bi.sah_cost, plain.sah_cost)


def test_closest_point_2m_faces(api, big):
    v, f, info, bvh, orc = big
    q = np.concatenate([near_surface_queries(v, f, 30000, seed=11), far_field_queries(v, 10000, seed=12)])
    qd = torch.as_tensor(q).cuda()
    d1, t1, b1 = api.closest_point(bvh, qd)
    d2, t2, b2 = api.closest_point_bruteforce(bvh, qd)                # same fp32 routine, every face
    assert torch.equal(d1, d2)
    same = (t1 == t2).float().mean().item()
    assert same > 0.995, same                                         # rest: reordered duplicates (near-ties)
    # oracle (fp64 brute force) on a sample, tie-free by its own gap filter
    idx = np.random.default_rng(0).choice(len(q), 1200, replace=False)
    r = orc.closest_points(q[idx])
    keep = (orc.runner_up(q[idx], r["tri"]) - r["dist"]) > 1e-4 * r["dist"]
    key = np.sort(f.astype(np.int64), axis=1)
    dup_of = {}
    tg = t1.cpu().numpy()[idx]
    same_face = np.array([np.array_equal(key[a], key[b]) for a, b in zip(tg, r["tri"])])
    assert keep.sum() > 600
    assert same_face[keep].all()                                      # the same triangle (possibly its duplicate)
    exact = tg == r["tri"]
    assert exact[keep].mean() > 0.98
    D = r["dist"]
    dg = d1.cpu().numpy()[idx]
    scale = float(np.abs(v).max())
    assert (np.abs(dg - D) <= 1e-6 * D + 2e-7 * scale).all()


@pytest.mark.parametrize("exterior", [False, True])
def test_walks_2m_faces_sampled_against_oracle(api, big, exterior):
    v, f, info, bvh, orc = big
    smp = fps_samples(v, f, 1500, n_candidates=60_000, seed=3)
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    # Kelvin origin: centre of the largest component's bounding box is inside that solid for these shapes
    comp = np.bincount(info["face_component"]).argmax()
    cv = v[np.unique(f[info["face_component"] == comp])]
    origin = tuple(float(x) for x in 0.5 * (cv.min(0) + cv.max(0)))
    kw = dict(seed=3, walks_per_sample=64, eps=1e-3, max_steps=512, include_killing=exterior,
              n_kill_walks=4096 if exterior else 0)
    gp = api.Params(kelvin_origin=origin, **kw)
    rec, steps, st = api.run_walks(bvh, S, gp, exterior, want_stats=True)
    rec2, steps2 = api.run_walks(bvh, S, gp, exterior)
    assert torch.equal(rec.view(torch.int32), rec2.view(torch.int32)) and torch.equal(steps, steps2)   # bitwise (tri_t = -1 is a NaN pattern)
    steps, rec = steps.cpu().numpy(), rec.cpu().numpy()
    assert st.n_truncated == int(((steps == -1) | (steps == -3)).sum()) and st.n_discarded * 64 == int((steps == -2).sum())
    assert (steps >= 0).mean() > 0.5                                  # flipped faces / overlaps cost some walks, not most
    ids = np.sort(np.random.default_rng(2).choice(len(smp["weight"]), 48, replace=False))
    n_w, n_kill = 4, 32
    orec = orc.run_walks_subset(OracleParams(origin=origin, **kw), exterior, smp["tri"], smp["bary"], smp["weight"],
                                ids, n_w, n_kill_first=n_kill)
    slots = (ids[:, None] * 64 + np.arange(n_w)[None, :]).ravel()
    if exterior:
        slots = np.concatenate([slots, len(smp["weight"]) * 64 + np.arange(n_kill)])
    # Flipped faces are NOT repaired here (no sidedness pre-pass), so some sampled walks start on the wrong side and are
    # cut by R10b / R10c or by max_steps on both sides; the outcome class must agree walk for walk.
    assert ((steps[slots] >= 0) == (orec["steps"] >= 0)).mean() >= 0.98
    same = steps[slots] == orec["steps"]
    assert same.mean() >= 0.95, (same.mean(), steps[slots], orec["steps"])
    ok = same & (steps[slots] >= 0)
    tri_t = rec[slots, 0].copy().view(np.int32)
    key = np.sort(f.astype(np.int64), axis=1)
    same_face = np.array([np.array_equal(key[a], key[b]) for a, b in zip(tri_t[ok], orec["tri_t"][ok])])
    assert same_face.mean() >= 0.95
    bt = np.stack([1 - rec[slots, 1] - rec[slots, 2], rec[slots, 1], rec[slots, 2]], 1).astype(np.float64)
    t_gpu = np.einsum("qk,qkd->qd", bt[ok], v[f[tri_t[ok]]].astype(np.float64))
    err = np.linalg.norm(t_gpu - orec["t"][ok], axis=1)
    assert np.quantile(err, 0.95) < 5e-4 and np.median(err) < 2e-5, np.quantile(err, [0.5, 0.95, 1.0])


@pytest.mark.parametrize("exterior", [False, True])
def test_walks_2m_faces_config3_size_bit_identical_reruns(api, big, exterior):
    """BASELINE config 3 at full size (20 000 FPS samples x 4096 walks = 82 M walks on the 2 M-face stress mesh): the
    records must not depend on the schedule.  Regression: with a purely relative pruning slack one walk in 82 M changed
    between reruns (near-tie between faces sharing an edge or vertex: the lane path and the warp-cooperative path visit
    the faces in different orders, and a face whose COMPUTED distance is the minimum was skipped when the other came
    first); fixed by the absolute margin of prune_limit (walk.cu)."""
    v, f, info, bvh, _ = big
    smp = fps_samples(v, f, 20_000, n_candidates=100_000, seed=3)
    S0 = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    nrm, _ = api.orient_samples(bvh, S0)
    S = api.Samples(S0.tri, S0.bary, S0.weight, nrm)
    comp = np.bincount(info["face_component"]).argmax()
    cv = v[np.unique(f[info["face_component"] == comp])]
    origin = tuple(float(x) for x in 0.5 * (cv.min(0) + cv.max(0)))
    P = api.Params(seed=0, walks_per_sample=4096, eps=1e-3, kelvin_origin=origin)
    rec0, steps0 = api.run_walks(bvh, S, P, exterior)
    r0 = rec0.view(torch.int32)
    for _ in range(5):
        rec, steps = api.run_walks(bvh, S, P, exterior)
        assert torch.equal(rec.view(torch.int32), r0) and torch.equal(steps, steps0)
        del rec, steps


def test_config3_sparse_matrix_entries_against_the_oracle_on_a_sample_subset(api):
    """BASELINE config 3 as bench.py builds it (2 M-face stress mesh, 20 000 FPS samples, Kelvin origin, sidedness
    pre-pass): every 1250th sample point (16 of 20 000, a 1/1250 subset) with 8 walks each, both operators, sparse
    output.  (1) The library's accumulation of the ORACLE's records equals the oracle's own accumulation (on the
    sub-mesh of touched faces: pure re-indexing) to fp32 rounding.  (2) The library's own walks + accumulation give
    entries within 4 Monte Carlo standard errors of the oracle's (same Philox counters, so in practice far closer)."""
    import argparse
    from bench import make_cfg3
    from oracle import RECORD_DTYPE
    args = argparse.Namespace(faces=2_000_000, components=30, samples=20_000, candidates=1_000_000, mesh_seed=3, no_cache=False)
    wl = make_cfg3(args)
    v, f = wl["v"], wl["f"]
    bvh = api.build_bvh(torch.as_tensor(v).cuda(), torch.as_tensor(f).cuda())
    ids = np.arange(0, len(wl["tri"]), 1250)
    tri, bary, wgt = wl["tri"][ids], wl["bary"][ids], wl["weight"][ids]
    S0 = api.Samples.from_arrays(tri, bary, wgt)
    nrm, _ = api.orient_samples(bvh, S0)
    S = api.Samples(S0.tri, S0.bary, S0.weight, nrm)
    nrm_h = nrm.cpu().numpy()
    orc = Oracle(mesh_geom(v, f))
    W = 8
    for exterior in (False, True):
        kw = dict(seed=0, walks_per_sample=W, eps=1e-3)
        P = api.Params(kelvin_origin=wl["origin"], **kw)
        orec, _ = orc.run_walks(OracleParams(origin=wl["origin"], **kw), exterior, tri, bary, wgt, normal=nrm_h)
        ok = orec["tri_t"] >= 0
        assert ok.mean() > 0.9
        # ---- sub-mesh of touched faces, oracle accumulation with variances
        faces_used = np.unique(np.concatenate([tri, orec["tri_t"][ok]]))
        verts_used, inv = np.unique(f[faces_used], return_inverse=True)
        f_sub = inv.reshape(-1, 3).astype(np.int32)
        face_new = -np.ones(len(f), np.int64); face_new[faces_used] = np.arange(len(faces_used))
        vert_new = -np.ones(len(v), np.int64); vert_new[verts_used] = np.arange(len(verts_used))
        sub = orec.copy()
        sub["tri_t"] = np.where(ok, face_new[np.maximum(orec["tri_t"], 0)], -1)
        osub = Oracle(mesh_geom(v[verts_used], f_sub))
        So, var = osub.accumulate_hat(sub, face_new[tri].astype(np.int32), bary, want_var=True)
        # ---- (1) the oracle's records through the library's sparse accumulation
        r = np.zeros((len(orec), 4), np.float32)
        r[:, 0] = np.where(ok, orec["tri_t"], -1).astype(np.int32).view(np.float32)
        r[:, 1], r[:, 2], r[:, 3] = orec["bary_t"][:, 1], orec["bary_t"][:, 2], np.where(ok, orec["weight"], 0.0)
        coo = api.accumulate_coo(bvh, S, P, torch.as_tensor(r).cuda())
        rr, cc = vert_new[coo.row.cpu().numpy()], vert_new[coo.col.cpu().numpy()]
        assert (rr >= 0).all() and (cc >= 0).all()
        Sg = np.zeros_like(So)
        Sg[rr, cc] = coo.val.cpu().numpy(); Sg[cc, rr] = coo.val.cpu().numpy()
        assert np.abs(Sg - So).max() <= 3e-5 * np.abs(So).max()
        # ---- (2) the library's own walks
        coo2, st = api.estimate_dtn_coo(bvh, S, P, exterior, want_stats=True)
        rec, steps = api.run_walks(bvh, S, P, exterior)
        same = steps.cpu().numpy() == orec["steps"]
        assert same.mean() >= 0.95, same.mean()
        r2, c2 = coo2.row.cpu().numpy(), coo2.col.cpu().numpy()
        inside = (vert_new[r2] >= 0) & (vert_new[c2] >= 0)
        S2 = np.zeros_like(So)
        S2[vert_new[r2[inside]], vert_new[c2[inside]]] = coo2.val.cpu().numpy()[inside]
        S2 = np.triu(S2) + np.triu(S2, 1).T
        se = np.sqrt(np.maximum(var, 0.0))
        scale = np.abs(So).max()
        bad = np.abs(S2 - So) > 4.0 * np.sqrt(2.0) * se + 2e-6 * scale
        assert bad.sum() <= max(1, int(1e-3 * (So != 0).sum())), (bad.sum(), (So != 0).sum())
        # entries of walks that ended elsewhere than the oracle's (a few per cent) fall outside the sub-mesh: small in norm
        out_norm = np.sqrt((coo2.val.cpu().numpy()[~inside].astype(np.float64) ** 2).sum())
        assert out_norm <= 0.2 * np.linalg.norm(So), (out_norm, np.linalg.norm(So))
        assert np.linalg.norm(S2 - So) <= np.linalg.norm(se) + 0.05 * np.linalg.norm(So)


def test_config3_in_the_bench_configuration_far_field_bounds_against_exact_queries(api):
    """BASELINE config 3 as bench.py times it: the 2 M-face stress mesh, 20 000 FPS samples, hierarchical sidedness,
    both operators in one sparse call, far-field lower bounds (interior far_alpha 1, exterior 2, near 2 eps), at the full
    4096 walks per sample.  Properties that hold at any size -- sorted upper-triangular entries without duplicates, the
    interior matrix annihilating constants, bit-identical reruns -- and the far-field estimator against the exact-query
    one on quadratic forms of smooth functions: 4 independent seeds each at 512 walks (same mean within the spread of the
    difference), and the two full-size runs within that spread scaled by sqrt(512 / 4096)."""
    import argparse
    import dataclasses
    from bench import make_cfg3
    args = argparse.Namespace(faces=2_000_000, components=30, samples=20_000, candidates=1_000_000, mesh_seed=3, no_cache=False)
    wl = make_cfg3(args)
    v = wl["v"]
    bvh = api.build_bvh(torch.as_tensor(v).cuda(), torch.as_tensor(wl["f"]).cuda())
    S0 = api.Samples.from_arrays(wl["tri"], wl["bary"], wl["weight"])
    nrm, _ = api.orient_samples_fast(bvh, S0, beta=2.5)
    S = api.Samples(S0.tri, S0.bary, S0.weight, nrm)
    far = (dict(far_alpha=1.0, far_near_factor=2.0), dict(far_alpha=2.0, far_near_factor=2.0))
    exact = (dict(), dict())
    xs = torch.as_tensor(np.stack([v[:, 0], v[:, 1], v[:, 2], v[:, 0] * v[:, 1], np.sin(3.0 * v[:, 2]), np.ones(len(v))], 1)).cuda().double()

    def run(kinds, W, seed, scratch):
        Pi = api.Params(seed=seed, walks_per_sample=W, eps=1e-3, **kinds[0])
        Pe = api.Params(seed=seed, walks_per_sample=W, eps=1e-3, kelvin_origin=wl["origin"], **kinds[1])
        return api.estimate_dtn_coo_both(bvh, S, Pi, Pe, scratch=scratch)

    def forms(coo):
        r, c, val = coo.row.long(), coo.col.long(), coo.val.double()
        w = torch.where(r == c, 1.0, 2.0).double() * val
        return (w[:, None] * xs[r] * xs[c]).sum(0).cpu().numpy()

    # ---- full size, the bench's own call
    sc = {}
    ci, ce = run(far, 4096, 0, sc)
    keep = [(m.row.clone(), m.col.clone(), m.val.clone()) for m in (ci, ce)]
    for m in (ci, ce):
        r, c = m.row.long(), m.col.long()
        assert m.nnz > 10_000_000 and bool((r <= c).all()) and int(c.max()) < len(v)
        key = r * len(v) + c
        assert bool((key[1:] > key[:-1]).all())                               # sorted by (row, col), one entry per position
        assert bool(torch.isfinite(m.val).all())
    q_far = [forms(ci), forms(ce)]
    # interior: S 1 = 0, row by row against the row's absolute sum
    r, c, val = ci.row.long(), ci.col.long(), ci.val.double()
    off = r != c
    rs = torch.zeros(len(v), dtype=torch.float64, device="cuda").index_add_(0, r, val).index_add_(0, c[off], val[off])
    ra = torch.zeros(len(v), dtype=torch.float64, device="cuda").index_add_(0, r, val.abs()).index_add_(0, c[off], val[off].abs())
    assert float((rs.abs() / ra.clamp_min(1e-30)).max()) < 1e-4
    assert abs(q_far[0][5]) < 1e-4 * float(ci.val.abs().sum())                # the constant's quadratic form
    ci2, ce2 = run(far, 4096, 0, sc)                                          # bit-identical rerun (same buffers: compare with the copies)
    for m, k in zip((ci2, ce2), keep):
        assert torch.equal(m.row, k[0]) and torch.equal(m.col, k[1]) and torch.equal(m.val, k[2])
    cxi, cxe = run(exact, 4096, 0, sc)
    q_exact = [forms(cxi), forms(cxe)]
    # ---- independent seeds at 512 walks: the two estimators have the same mean
    R = 4
    qf = np.array([[forms(m) for m in run(far, 512, 100 + s, sc)] for s in range(R)])        # [R][2][6]
    qx = np.array([[forms(m) for m in run(exact, 512, 200 + s, sc)] for s in range(R)])
    sd = np.sqrt(qf.std(0, ddof=1) ** 2 + qx.std(0, ddof=1) ** 2)                               # spread of one difference
    scale = np.abs(qx.mean(0)) + 1e-12
    for op in range(2):
        for k in range(5):                                                                      # the five non-constant functions
            assert abs(qf[:, op, k].mean() - qx[:, op, k].mean()) <= 5.0 * sd[op, k] / np.sqrt(R) + 1e-3 * scale[op, k], (op, k)
            # full size, same seed in both runs: inside the spread of two independent full-size runs
            assert abs(q_far[op][k] - q_exact[op][k]) <= 5.0 * sd[op, k] * np.sqrt(512.0 / 4096.0) + 1e-3 * scale[op, k], (op, k)
