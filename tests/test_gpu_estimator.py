"""GPU parity, estimator half: tangent balls, per-walk records, the deterministic
accumulation, and the assembled interior / exterior DtN matrices against the CPU
oracle (same Philox streams, brute-force fp64 geometry).  Bars (BASELINE.json
north_star): matrix entries within 4 Monte Carlo standard errors of the oracle,
identical seeds bit-identical run to run, exact symmetry, zero row sums for the
interior operator.  Everything goes through the C ABI."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import Oracle, OracleParams, mesh_geom, steklov_eigs              # noqa: E402
from synth import (box, icosphere, merge_meshes, stress_mesh, torus,            # noqa: E402
                   uniform_samples, vertex_cell_samples)


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


def _cuda(a, dtype):
    return torch.as_tensor(np.ascontiguousarray(a)).to(device="cuda", dtype=dtype)


def _setup(api, v, f, smp):
    bvh = api.build_bvh(_cuda(v, torch.float32), _cuda(f, torch.int32))
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    return bvh, S


def _params(api, **kw):
    g = dict(kw)
    o = dict(kw)
    if "kelvin_origin" in g:
        o["origin"] = o.pop("kelvin_origin")
    return api.Params(**g), OracleParams(**o)


def _unpack_records(rec):
    r = rec.cpu().numpy()
    return r[:, 0].copy().view(np.int32), r[:, 1], r[:, 2], r[:, 3]


# ------------------------------------------------------------------------------
# A2: tangent balls
# ------------------------------------------------------------------------------
@pytest.mark.parametrize("exterior", [False, True])
def test_tangent_balls_match_oracle(api, exterior):
    v, f = merge_meshes([icosphere(3), box((0.6, 0.8, 1.0), (3, 3, 3), center=(1.4, 0.2, 0.0))])[:2]
    smp = uniform_samples(v, f, 3000, seed=4)
    bvh, S = _setup(api, v, f, smp)
    P, OP = _params(api, eps=1e-4, walks_per_sample=1, max_steps=0, kelvin_origin=(0.1, 0.05, -0.1))
    balls = api.tangent_balls(bvh, S, P, exterior).cpu().numpy()
    _, ob = Oracle(mesh_geom(v, f)).run_walks(OP, exterior, smp["tri"], smp["bary"], smp["weight"])
    r_gpu, r_orc = balls[:, 3], ob[:, 0]
    # the bisection takes the same branch unless a probe distance is within fp32 rounding of
    # its threshold; then the two radii differ by one bisection cell at some level
    same = np.abs(r_gpu - r_orc) <= 2e-6 * np.maximum(r_orc, 1e-3)
    assert same.mean() > 0.995, same.mean()
    assert np.abs(balls[same][:, :3] - ob[same][:, 1:4]).max() < 5e-6
    if exterior:
        assert np.abs(balls[:, 7] - ob[:, 4]).max() < 1e-5 * ob[:, 4].max()
    assert ((r_gpu > 0) == (r_orc > 0)).mean() > 0.995


# ------------------------------------------------------------------------------
# A3-A6: per-walk records.  fp32 vs fp64 walks follow the same Philox stream, so
# nearly every walk takes the same number of jumps and lands at the same point.
# ------------------------------------------------------------------------------
def _compare_records(api, v, f, smp, exterior, gp, op, min_same=0.97):
    bvh, S = _setup(api, v, f, smp)
    rec, steps, st = api.run_walks(bvh, S, gp, exterior, want_stats=True)
    tri_t, b1, b2, wgt = _unpack_records(rec)
    steps = steps.cpu().numpy()
    orc = Oracle(mesh_geom(v, f))
    orec, _ = orc.run_walks(op, exterior, smp["tri"], smp["bary"], smp["weight"])
    assert len(orec) == len(steps)
    # statistics kept by the kernel agree with what it wrote
    assert st.n_walks == len(steps)
    assert st.n_truncated == int((steps == -1).sum()) + int((steps == -3).sum())     # -3: left the AABB (R10b)
    assert st.n_steps >= int(steps[steps > 0].sum()) + int((steps == -1).sum()) * gp.max_steps
    assert st.n_steps <= int(steps[steps > 0].sum()) + int(((steps == -1) | (steps == -3)).sum()) * gp.max_steps
    same = steps == orec["steps"]
    assert same.mean() >= min_same, same.mean()
    ok = same & (steps >= 0)
    # exit point: same place on the surface
    bt = np.stack([1 - b1 - b2, b1, b2], 1).astype(np.float64)
    t_gpu = np.einsum("qk,qkd->qd", bt[ok], v[f[tri_t[ok]]].astype(np.float64))
    err = np.linalg.norm(t_gpu - orec["t"][ok], axis=1)
    scale = float(np.abs(v).max())
    assert np.quantile(err, 0.99) < 2e-4 * scale, np.quantile(err, [0.5, 0.99, 1.0])
    same_tri = tri_t[ok] == orec["tri_t"][ok]
    assert same_tri.mean() > 0.98
    rel = np.abs(wgt[ok] - orec["weight"][ok]) / np.abs(orec["weight"][ok]).max()
    assert np.quantile(rel, 0.99) < 1e-4
    # distribution of walk lengths (all walks, diverged ones included)
    g, o = steps[steps >= 0], orec["steps"][orec["steps"] >= 0]
    assert abs(g.mean() - o.mean()) < 0.03 * max(o.mean(), 1.0)
    return rec, steps, orec, st


def test_interior_records_match_oracle_icosphere(api):
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 4, seed=0)
    gp, op = _params(api, seed=11, walks_per_sample=64, eps=1e-3)
    _compare_records(api, v, f, smp, False, gp, op)


def test_interior_records_uniform_antithetic_multi_component(api):
    v, f = merge_meshes([icosphere(3), box((0.6, 0.8, 1.0), (3, 3, 3), center=(2.4, 0.2, 0.0)),
                         torus(1.0, 0.3, 40, 20, axis="z", center=(0, 0, 3.0))])[:2]
    smp = uniform_samples(v, f, 400, seed=9)
    gp, op = _params(api, seed=3, walks_per_sample=32, eps=1e-4, importance_sample=False, antithetic=True)
    _compare_records(api, v, f, smp, False, gp, op)


@pytest.mark.parametrize("origin", [(0.0, 0.0, 0.0), (0.3, 0.1, -0.2)])
def test_exterior_records_and_killing_match_oracle(api, origin):
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 2, seed=1)
    gp, op = _params(api, seed=5, walks_per_sample=64, eps=1e-3, include_killing=True, n_kill_walks=5000,
                     kelvin_origin=origin)
    rec, steps, orec, st = _compare_records(api, v, f, smp, True, gp, op)
    n_main = len(smp["weight"]) * 64
    assert len(steps) == n_main + 5000
    # capacity of the (polyhedral) unit sphere from the killing walks: sum of weights = 4 pi E|t0|
    wk = _unpack_records(rec)[3][n_main:]
    assert abs(wk.sum() / (4 * np.pi) - 1.0) < 0.02


def test_truncated_and_discarded_walks(api):
    """max_steps cuts walks (counted, weightless); flipped normals put the tangent ball
    outside: on a closed convex solid those walks never return and are truncated."""
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 1, seed=2)
    bvh, S = _setup(api, v, f, smp)
    gp, op = _params(api, seed=1, walks_per_sample=16, eps=1e-5, max_steps=3)
    rec, steps, st = api.run_walks(bvh, S, gp, False, want_stats=True)
    orec, _ = Oracle(mesh_geom(v, f)).run_walks(op, False, smp["tri"], smp["bary"], smp["weight"])
    steps = steps.cpu().numpy()
    assert (steps == -1).sum() > 0 and st.n_truncated == (steps == -1).sum()
    assert ((steps == -1) == (orec["steps"] == -1)).mean() > 0.98
    tri_t, _, _, wgt = _unpack_records(rec)
    assert (tri_t[steps == -1] == -1).all() and (wgt[steps == -1] == 0).all()
    # zero-radius balls: normal override pointing along the surface -> every probe hits
    nrm = np.zeros((len(smp["weight"]), 3), np.float32)
    S2 = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"], normal=nrm)
    rec, steps, st = api.run_walks(bvh, S2, api.Params(walks_per_sample=2, eps=1e-3), False, want_stats=True)
    assert st.n_discarded == len(smp["weight"]) and (steps.cpu().numpy() == -2).all()


# ------------------------------------------------------------------------------
# A7: deterministic accumulation
# ------------------------------------------------------------------------------
def test_accumulate_from_oracle_records_matches_oracle_matrix(api):
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 3, seed=3)
    orc = Oracle(mesh_geom(v, f))
    op = OracleParams(seed=2, walks_per_sample=32, eps=1e-3, include_killing=True, n_kill_walks=3000)
    out = orc.estimate_dtn(op, True, smp["tri"], smp["bary"], smp["weight"])
    orec = out["records"]
    rec = np.zeros((len(orec), 4), np.float32)
    rec[:, 0] = orec["tri_t"].astype(np.int32).view(np.float32)
    rec[:, 1] = orec["bary_t"][:, 1]
    rec[:, 2] = orec["bary_t"][:, 2]
    rec[:, 3] = orec["weight"]
    bvh, S = _setup(api, v, f, smp)
    gp = api.Params(seed=2, walks_per_sample=32, eps=1e-3, include_killing=True, n_kill_walks=3000)
    Sg, st = api.accumulate(bvh, S, gp, _cuda(rec, torch.float32), want_stats=True)
    Sg = Sg.cpu().numpy().astype(np.float64)
    So = out["S"]
    # fp32 sums of ~1e2..1e4 terms per entry
    assert np.abs(Sg - So).max() <= 3e-5 * np.abs(So).max()
    assert np.array_equal(Sg, Sg.T)
    assert st.n_unique <= st.n_entries and st.n_unique >= np.count_nonzero(np.triu(So))
    # run to run bit identity
    Sg2 = api.accumulate(bvh, S, gp, _cuda(rec, torch.float32)).cpu().numpy()
    assert np.array_equal(Sg2.astype(np.float64), Sg)


# ------------------------------------------------------------------------------
# The assembled matrices
# ------------------------------------------------------------------------------
def _hit_counts(out, smp, f, K):
    """Number of oracle walks that contribute to each matrix entry (hat basis: the vertices
    of the sample's face and of the exit face)."""
    rec = out["records"]
    ok = (rec["steps"] >= 0) & (rec["weight"] != 0)
    r = rec[ok]
    main = r["sample"] >= 0
    vt = f[r["tri_t"]].astype(np.int64)
    vs = np.where(main[:, None], f[np.asarray(smp["tri"])[np.maximum(r["sample"], 0)]].astype(np.int64), vt)
    idx = np.concatenate([vs, vt], 1)
    cnt = np.zeros((K, K), np.int64)
    for p in range(6):
        for q in range(6):
            new = np.ones(len(idx), bool)                 # count each (row, col) once per walk
            for p2 in range(6):
                for q2 in range(6):
                    if (p2, q2) < (p, q):
                        new &= ~((idx[:, p2] == idx[:, p]) & (idx[:, q2] == idx[:, q]))
            np.add.at(cnt, (idx[new, p], idx[new, q]), 1)
    return cnt


def _assert_within_4se(Sg, out, smp, f, min_hits=32):
    """BASELINE north_star: entries within 4 Monte Carlo standard errors of the oracle, on
    entries with >= 32 contributing walks; the variance estimate of an
    entry hit by a handful of walks says nothing.  The same Philox streams make the two
    far closer than that overall: Frobenius difference below one standard error."""
    So, var = out["S"], out["var"]
    cnt = _hit_counts(out, smp, f, len(So))
    se = np.sqrt(2.0 * var)                             # both sides carry the same Monte Carlo error
    scale = np.abs(So).max()
    sel = cnt >= min_hits
    assert sel.sum() > 100
    bad = (np.abs(Sg - So) > 4.0 * se + 2e-6 * scale) & sel
    assert bad.sum() <= max(1, int(1e-4 * sel.sum())), (bad.sum(), sel.sum())
    assert np.linalg.norm(Sg - So) <= np.linalg.norm(np.sqrt(var))


def test_config0_interior_icosphere_l2(api):
    """BASELINE config 0: icosphere L2, hat basis, 1024 walks per vertex (G = 8 sample points
    per vertex x 128 walks), eps 1e-3, cap 2.5 deg, seed 0."""
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 8, seed=0)
    gp, op = _params(api, seed=0, walks_per_sample=128, eps=1e-3)
    bvh, S = _setup(api, v, f, smp)
    Sg, st = api.estimate_dtn_interior(bvh, S, gp, want_stats=True)
    Sg2 = api.estimate_dtn_interior(bvh, S, gp)
    assert torch.equal(Sg, Sg2)                          # bit-identical run to run
    Sg = Sg.cpu().numpy().astype(np.float64)
    assert st.n_walks == 162 * 1024 and st.n_truncated == 0
    assert np.array_equal(Sg, Sg.T)                      # exactly symmetric
    assert np.abs(Sg.sum(1)).max() < 2e-5 * np.abs(Sg).max()     # annihilates constants
    orc = Oracle(mesh_geom(v, f))
    out = orc.estimate_dtn(op, False, smp["tri"], smp["bary"], smp["weight"], want_var=True)
    _assert_within_4se(Sg, out, smp, f)
    # spectrum: 0, 1 (x3), 2 (x5), 3 (x7) up to the cap / eps / mesh bias stated in DESIGN.md
    M = orc.mass_matrix()
    lam_g, lam_o = steklov_eigs(Sg, M, 16), steklov_eigs(out["S"], M, 16)
    assert abs(lam_g[0]) < 1e-4
    assert np.abs(lam_g - lam_o).max() < 0.03
    for l, sl in ((1, slice(1, 4)), (2, slice(4, 9)), (3, slice(9, 16))):
        assert abs(lam_g[sl].mean() / l - 1) < 0.12, (l, lam_g[sl])
    assert np.linalg.eigvalsh(Sg).min() > -1e-5 * np.abs(Sg).max()          # PSD


def test_exterior_with_killing_icosphere_l2(api):
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 4, seed=0)
    gp, op = _params(api, seed=7, walks_per_sample=128, eps=1e-3, include_killing=True,
                     n_kill_walks=162 * 512, kelvin_origin=(0.2, -0.1, 0.1))
    bvh, S = _setup(api, v, f, smp)
    Sg, st = api.estimate_dtn_exterior(bvh, S, gp, want_stats=True)
    assert torch.equal(Sg, api.estimate_dtn_exterior(bvh, S, gp))
    Sg = Sg.cpu().numpy().astype(np.float64)
    assert np.array_equal(Sg, Sg.T)
    orc = Oracle(mesh_geom(v, f))
    out = orc.estimate_dtn(op, True, smp["tri"], smp["bary"], smp["weight"], want_var=True)
    _assert_within_4se(Sg, out, smp, f)
    M = orc.mass_matrix()
    lam = steklov_eigs(Sg, M, 9)
    assert abs(lam[0] - 1.0) < 0.08                      # l + 1 with l = 0
    assert abs(lam[1:4].mean() - 2.0) < 0.2
    # killing off: constants are annihilated again
    gp.include_killing = False
    S0 = api.estimate_dtn_exterior(bvh, S, gp).cpu().numpy().astype(np.float64)
    assert np.abs(S0.sum(1)).max() < 5e-5 * np.abs(S0).max()


def test_interior_does_not_couple_components_exterior_does(api):
    """PAPER.md:50, 303-309; SURVEY.md 8(c) 'Coupling'."""
    va, fa = icosphere(2, 1.0, (-1.25, 0, 0))
    vb, fb = icosphere(2, 1.0, (+1.25, 0, 0))
    v, f = merge_meshes([(va, fa), (vb, fb)])[:2]
    smp = vertex_cell_samples(v, f, 2, seed=0)
    bvh, S = _setup(api, v, f, smp)
    gp = api.Params(seed=1, walks_per_sample=64, eps=1e-3, kelvin_origin=(-1.25, 0, 0))
    nA = len(va)
    Si = api.estimate_dtn_interior(bvh, S, gp).cpu().numpy()
    assert (Si[:nA, nA:] == 0).all() and (Si[nA:, :nA] == 0).all()
    Se = api.estimate_dtn_exterior(bvh, S, gp).cpu().numpy()
    assert np.linalg.norm(Se[:nA, nA:]) > 1e-3 * np.linalg.norm(Se)


def test_stress_mesh_subset_against_oracle(api):
    """In-the-wild style mesh (slivers, duplicates, flips, many components): records agree
    with the brute-force oracle walk for walk; the matrix is symmetric and reproducible."""
    v, f, info = stress_mesh(n_faces=6000, n_components=6, seed=3)
    smp = uniform_samples(v, f, 256, seed=8)
    gp, op = _params(api, seed=4, walks_per_sample=16, eps=1e-3, max_steps=256)
    _compare_records(api, v, f, smp, False, gp, op, min_same=0.95)
    bvh, S = _setup(api, v, f, smp)
    A = api.estimate_dtn_interior(bvh, S, gp)
    assert torch.equal(A, api.estimate_dtn_interior(bvh, S, gp)) and torch.equal(A, A.T)


def test_exterior_on_a_leaky_mesh_cuts_inside_walkers(api):
    """Regression + R10c.  A noise-displaced sphere with slivers, duplicates and flipped faces (config 3/4 style):
    exterior walks that start on the wrong side of a flipped face run inside the solid, where the Kelvin
    coordinate doubles per jump.  They are cut (-3) as soon as their empty ball holds the inversion centre; no
    walk overflows, whole-tree queries are completed by the warp (this mesh once broke that path), and sampled
    walks agree with the oracle walk for walk."""
    from synth import fps_samples
    v, f, info = stress_mesh(n_faces=52410, n_components=1, seed=100)
    smp = fps_samples(v, f, 512, n_candidates=12000, seed=0)
    origin = tuple(float(x) for x in 0.5 * (v.min(0) + v.max(0)))
    bvh, S = _setup(api, v, f, smp)
    W = 256
    kw = dict(seed=1, walks_per_sample=W, eps=1e-3, max_steps=512, include_killing=True, n_kill_walks=4096)
    gp = api.Params(kelvin_origin=origin, **kw)
    rec, steps, st = api.run_walks(bvh, S, gp, True, want_stats=True)
    rec2, steps2 = api.run_walks(bvh, S, gp, True)
    assert torch.equal(rec.view(torch.int32), rec2.view(torch.int32)) and torch.equal(steps, steps2)
    steps = steps.cpu().numpy()
    assert st.n_truncated == int(((steps == -1) | (steps == -3)).sum())
    assert (steps == -3).sum() > 0 and (steps == -1).mean() < 1e-3
    assert st.n_steps < 40 * len(steps)                               # no walker runs for hundreds of doubling jumps
    ids = np.sort(np.random.default_rng(5).choice(512, 24, replace=False))
    n_w, n_kill = 4, 16
    orec = Oracle(mesh_geom(v, f)).run_walks_subset(OracleParams(origin=origin, **kw), True, smp["tri"], smp["bary"],
                                                     smp["weight"], ids, n_w, n_kill_first=n_kill)
    slots = np.concatenate([(ids[:, None] * W + np.arange(n_w)[None, :]).ravel(), 512 * W + np.arange(n_kill)])
    same = steps[slots] == orec["steps"]
    assert same.mean() >= 0.9, (same.mean(), steps[slots], orec["steps"])
    A = api.estimate_dtn_coo(bvh, S, gp, exterior=True)
    assert A.nnz > 0


def test_estimator_argument_errors(api):
    v, f = icosphere(1)
    smp = vertex_cell_samples(v, f, 1, seed=0)
    bvh, S = _setup(api, v, f, smp)
    for bad in (dict(eps=0.0), dict(walks_per_sample=0), dict(cap_half_angle_deg=0.0), dict(bisection_iters=0)):
        with pytest.raises(api.McsError) as e:
            api.estimate_dtn_interior(bvh, S, api.Params(**{**dict(walks_per_sample=2), **bad}))
        assert e.value.code == api.MCS_EINVAL
    with pytest.raises(api.McsError) as e:                # workspace too small
        api.estimate_dtn_interior(bvh, S, api.Params(walks_per_sample=2), workspace=torch.empty(16, dtype=torch.uint8, device="cuda"),
                                  _exact_workspace=True)
    assert e.value.code == api.MCS_ENOMEM
    badS = api.Samples.from_arrays(np.full_like(smp["tri"], len(f)), smp["bary"], smp["weight"])
    with pytest.raises(api.McsError) as e:                # sample face out of range
        api.estimate_dtn_interior(bvh, badS, api.Params(walks_per_sample=2))
    assert e.value.code == api.MCS_EINVAL
    with pytest.raises(api.McsError) as e:                # Kelvin origin on a vertex
        api.estimate_dtn_exterior(bvh, S, api.Params(walks_per_sample=2, kelvin_origin=tuple(float(x) for x in v[0])))
    assert e.value.code == api.MCS_EDEGENERATE


def test_config2a_two_spheres_capacity_and_coupling_decay(api):
    """BASELINE config 2 (spheres-only variant 2a, SURVEY.md 8(c) 'Killing / escape', 'Coupling'):
    the killing term sums to 4 pi * capacity; two unit spheres with centres 2.5 apart have capacity
    1.4553 (classical image series 2 a sinh(beta) sum_n (-1)^(n+1) / sinh(n beta), cosh(beta) = d / 2a);
    the exterior coupling block decays with the separation, the interior one is exactly zero."""
    def series(d, a=1.0, n=200):
        beta = np.arccosh(d / (2 * a))
        k = np.arange(1, n + 1)
        return 2 * a * np.sinh(beta) * np.sum((-1.0) ** (k + 1) / np.sinh(k * beta))
    assert abs(series(2.5) - 1.4553) < 2e-4
    norms = []
    for d in (2.5, 3.0, 4.0, 6.0):
        level = 3
        va, fa = icosphere(level, 1.0, (-d / 2, 0, 0))
        vb, fb = icosphere(level, 1.0, (+d / 2, 0, 0))
        v, f = merge_meshes([(va, fa), (vb, fb)])[:2]
        smp = vertex_cell_samples(v, f, 2, seed=0)
        bvh, S = _setup(api, v, f, smp)
        nA = len(va)
        P = api.Params(seed=3, walks_per_sample=128, eps=1e-3, include_killing=True, n_kill_walks=400_000,
                       kelvin_origin=(-d / 2, 0, 0))
        Se = api.estimate_dtn_exterior(bvh, S, P).cpu().numpy().astype(np.float64)
        cap = Se.sum() / (4 * np.pi)                     # jump part annihilates constants
        assert abs(cap / series(d) - 1) < 0.02, (d, cap, series(d))     # polyhedral spheres + 4e5 walks
        # total weight of the walks that start on one sphere and exit on the other (a sum: robust to MC noise)
        norms.append(-Se[:nA, nA:].sum() / np.trace(Se[:nA, :nA]))
        if d == 2.5:
            Si = api.estimate_dtn_interior(bvh, S, api.Params(seed=3, walks_per_sample=128, eps=1e-3)).cpu().numpy()
            assert (Si[:nA, nA:] == 0).all()
    assert norms[0] > norms[1] > norms[2] > norms[3] > 0, norms


def test_w1_many_samples_per_chunk_and_odd_sizes(api):
    """Alg. 2 as printed: one walk per sample (W = 1), so a level-1 block of the accumulation holds 256
    different samples; odd counts exercise the ragged tails (samples, walks, killing walks)."""
    v, f = icosphere(2)
    smp = uniform_samples(v, f, 3001, seed=13)
    gp, op = _params(api, seed=21, walks_per_sample=1, eps=1e-3, include_killing=True, n_kill_walks=777,
                     kelvin_origin=(0.05, 0.1, 0.0))
    bvh, S = _setup(api, v, f, smp)
    orc = Oracle(mesh_geom(v, f))
    for ext in (False, True):
        fn = api.estimate_dtn_exterior if ext else api.estimate_dtn_interior
        Sg = fn(bvh, S, gp)
        assert torch.equal(Sg, fn(bvh, S, gp)) and torch.equal(Sg, Sg.T)
        out = orc.estimate_dtn(op, ext, smp["tri"], smp["bary"], smp["weight"], want_var=True)
        Sg = Sg.cpu().numpy().astype(np.float64)
        assert np.linalg.norm(Sg - out["S"]) <= np.linalg.norm(np.sqrt(out["var"]))
        # the library's accumulation of its own records equals the oracle's accumulation of them
        rec, steps = api.run_walks(bvh, S, gp, ext)
        r = rec.cpu().numpy()
        from oracle import RECORD_DTYPE
        orec = np.zeros(len(r), RECORD_DTYPE)
        tri_t = r[:, 0].copy().view(np.int32)
        n_main = len(smp["tri"])
        orec["sample"] = np.where(np.arange(len(r)) < n_main, np.arange(len(r)), -1)
        orec["tri_t"] = tri_t
        orec["bary_t"][:, 1] = r[:, 1]; orec["bary_t"][:, 2] = r[:, 2]
        orec["bary_t"][:, 0] = 1.0 - r[:, 1].astype(np.float32) - r[:, 2].astype(np.float32)
        orec["weight"] = np.where(tri_t >= 0, r[:, 3], 0.0)
        orec["steps"] = np.where(tri_t >= 0, 0, -1)
        So = orc.accumulate_hat(orec, smp["tri"], smp["bary"])
        assert np.abs(Sg - So).max() <= 3e-5 * np.abs(So).max()


def test_tiny_meshes_and_normal_override(api):
    """A tetrahedron (4 faces) runs the whole path; an explicit normal array equal to the face normals gives
    the same matrix bit for bit."""
    v = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1]], np.float32)
    f = np.array([[0, 2, 1], [0, 1, 3], [0, 3, 2], [1, 2, 3]], np.int32)          # outward winding
    smp = uniform_samples(v, f, 64, seed=2)
    bvh, S = _setup(api, v, f, smp)
    P = api.Params(seed=5, walks_per_sample=32, eps=1e-3)
    A, st = api.estimate_dtn_interior(bvh, S, P, want_stats=True)
    assert st.n_truncated == 0 and torch.equal(A, A.T)
    Sg = A.cpu().numpy().astype(np.float64)
    assert np.abs(Sg.sum(1)).max() < 5e-5 * np.abs(Sg).max() and np.linalg.eigvalsh(Sg).min() > -1e-5 * np.abs(Sg).max()
    vv = v[f[smp["tri"]]].astype(np.float64)
    nrm = np.cross(vv[:, 1] - vv[:, 0], vv[:, 2] - vv[:, 0]).astype(np.float32)
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    S2 = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"], normal=nrm)
    B = api.estimate_dtn_interior(bvh, S2, P)
    assert (A - B).abs().max().item() <= 1e-5 * A.abs().max().item()


# ------------------------------------------------------------------------------
# Alg. 1, the naive finite-difference estimator
# ------------------------------------------------------------------------------
def test_naive_estimator_records_and_matrix_match_oracle(api):
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 4, seed=0)
    gp, op = _params(api, seed=6, walks_per_sample=64, eps=1e-4, estimator=1, inset=0.02)
    rec, steps, orec, st = _compare_records(api, v, f, smp, False, gp, op)
    assert st.n_discarded == 0 and (steps >= 1).all()                   # the inset point is outside the shell
    bvh, S = _setup(api, v, f, smp)
    A = api.estimate_dtn_interior(bvh, S, gp)
    assert torch.equal(A, api.estimate_dtn_interior(bvh, S, gp)) and torch.equal(A, A.T)
    Sg = A.cpu().numpy().astype(np.float64)
    out = Oracle(mesh_geom(v, f)).estimate_dtn(op, False, smp["tri"], smp["bary"], smp["weight"], want_var=True)
    _assert_within_4se(Sg, out, smp, f)
    assert np.linalg.eigvalsh(Sg).min() < -1e-3 * np.abs(Sg).max()      # PSD only in expectation (PAPER.md, after Eq. 16)
    coo = api.estimate_dtn_coo(bvh, S, gp, False)
    assert torch.equal(coo.to_dense(), A)
    with pytest.raises(api.McsError) as e:                               # Alg. 1 is the interior estimator
        api.estimate_dtn_exterior(bvh, S, gp)
    assert e.value.code == api.MCS_EINVAL
    with pytest.raises(api.McsError):
        api.estimate_dtn_interior(bvh, S, api.Params(walks_per_sample=2, estimator=1, inset=0.0))


# ------------------------------------------------------------------------------
# both operators in one call (mcs_estimate_dtn_both): walk kernels overlapped on two streams
# ------------------------------------------------------------------------------
@pytest.mark.parametrize("case", ["sphere", "components"])
def test_both_operators_in_one_call_equal_the_single_calls_bit_for_bit(api, case):
    if case == "sphere":
        v, f = icosphere(3)
        smp = vertex_cell_samples(v, f, 4, seed=2)
        W, kill = 64, 4096
    else:
        v, f = merge_meshes([icosphere(2), torus(1.0, 0.3, 24, 12, center=(3.0, 0.0, 0.0)),
                             box((0.6, 0.8, 1.0), (3, 3, 3), center=(0.0, 2.5, 0.0))])[:2]
        smp = uniform_samples(v, f, 1777, seed=9)
        W, kill = 37, 5001
    bvh, S = _setup(api, v, f, smp)
    Pi = api.Params(seed=11, walks_per_sample=W, eps=1e-3)
    Pe = api.Params(seed=12, walks_per_sample=W, eps=1e-3, include_killing=True, n_kill_walks=kill,
                    kelvin_origin=(0.05, -0.02, 0.03))
    Si = api.estimate_dtn_interior(bvh, S, Pi).clone()
    Se = api.estimate_dtn_exterior(bvh, S, Pe).clone()
    Bi, Be, st_i, st_e = api.estimate_dtn_both(bvh, S, Pi, Pe, want_stats=True)
    assert torch.equal(Bi, Si) and torch.equal(Be, Se)
    assert st_i.n_walks == S.n_s * W and st_e.n_walks == S.n_s * W + kill
    assert st_i.n_steps > 0 and st_e.n_steps > 0
    # again without the counters (the instance bench.py times), on a side stream, several times in a row
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        for _ in range(3):
            Ci, Ce = api.estimate_dtn_both(bvh, S, Pi, Pe)
            # work queued behind the call on the caller's stream sees both results
            di, de = (Ci - Si).abs().max(), (Ce - Se).abs().max()
    side.synchronize()
    assert float(di) == 0.0 and float(de) == 0.0


def test_both_operators_argument_errors(api):
    v, f = icosphere(1)
    smp = vertex_cell_samples(v, f, 2, seed=0)
    bvh, S = _setup(api, v, f, smp)
    P = api.Params(seed=1, walks_per_sample=8, eps=1e-3)
    out = torch.empty((bvh.V, bvh.V), dtype=torch.float32, device="cuda")
    with pytest.raises(api.McsError):          # the operators run concurrently: one buffer for both is refused
        api.estimate_dtn_both(bvh, S, P, P, out_interior=out, out_exterior=out)
    need = api.workspace_bytes_both(bvh, S, P, P)
    assert need == api.workspace_bytes(bvh, S, P, False) + api.workspace_bytes(bvh, S, P, True)


@pytest.mark.parametrize("ops", [(True, False), (False, True), (True, True)])
def test_host_entry_point_equals_the_device_calls_bit_for_bit(api, ops):
    """mcs_estimate_dtn_host (upload, build, estimate, download; with both operators: the overlapped call with each
    download on its operator's stream) against build_bvh + estimate_dtn_* on device tensors."""
    interior, exterior = ops
    v, f = merge_meshes([icosphere(2), box((0.6, 0.8, 1.0), (3, 3, 3), center=(2.2, 0.1, 0.0))])[:2]
    smp = uniform_samples(v, f, 1501, seed=3)
    bvh, S = _setup(api, v, f, smp)
    P = api.Params(seed=5, walks_per_sample=48, eps=1e-3, include_killing=True, n_kill_walks=7777,
                   kelvin_origin=(0.02, 0.01, -0.03))
    res = api.estimate_dtn_host(torch.as_tensor(v, dtype=torch.float32), torch.as_tensor(f, dtype=torch.int32),
                                torch.as_tensor(smp["tri"]), torch.as_tensor(smp["bary"]), torch.as_tensor(smp["weight"]),
                                P, interior=interior, exterior=exterior, want_stats=True)
    if interior:
        assert torch.equal(res["interior"], api.estimate_dtn_interior(bvh, S, P).cpu())
    if exterior:
        assert torch.equal(res["exterior"], api.estimate_dtn_exterior(bvh, S, P).cpu())
        assert res["stats"].n_walks == S.n_s * 48 + 7777
    assert res["d2h_bytes"] == (int(interior) + int(exterior)) * bvh.V * bvh.V * 4


def test_handle_freed_while_work_is_queued_on_a_side_stream(api):
    """mcs_free_bvh must order the release of the tree's memory after the last call that used the handle, also when that
    call ran on a NON-BLOCKING stream (PyTorch's side streams), which the legacy default stream does not wait for: the
    handle records an event on the stream of every call and the free waits for it.  Estimate on a side stream, drop the
    handle at once, immediately build other trees (which reuse the pool's memory), and compare with an undisturbed run."""
    v, f = icosphere(3)
    smp = vertex_cell_samples(v, f, 4, seed=1)
    vd, fd = torch.as_tensor(v).cuda(), torch.as_tensor(f).cuda()
    S = api.Samples.from_arrays(smp["tri"], smp["bary"], smp["weight"])
    P = api.Params(seed=3, walks_per_sample=256, eps=1e-4)
    ref = api.estimate_dtn_interior(api.build_bvh(vd, fd), S, P).clone()
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    for _ in range(8):
        with torch.cuda.stream(side):
            bvh = api.build_bvh(vd, fd)
            out = api.estimate_dtn_interior(bvh, S, P)
            del bvh                                                   # freed while the accumulation may still be queued
            junk = [api.build_bvh(vd * 1.5, fd) for _ in range(3)]    # grabs memory from the pool right away
            del junk
        side.synchronize()
        assert torch.equal(out, ref)
