"""Pins for the oracle's estimator pieces against what the paper and the
mathematics fix (no GPU): tangent balls, walk-on-spheres harmonic-measure
identities, the analytic-ball spectra l (interior) and l+1 (exterior, centred
and off-centre), capacity, and the structural invariants on meshes."""
import numpy as np
import pytest
from scipy.integrate import quad
from scipy.special import eval_legendre

from oracle import Oracle, OracleParams, mesh_geom, sphere_geom, steklov_eigs
from synth import box, icosphere, merge_meshes, uniform_samples, vertex_cell_samples

from sph import DEGREES, fibonacci_sphere, real_sph_harm


# --------------------------------------------------------------------------
# tangent balls
# --------------------------------------------------------------------------
def test_tangent_ball_interior_sphere_closed_form():
    orc = Oracle(sphere_geom((0.1, -0.2, 0.3), 2.0))
    pos = fibonacci_sphere(32) * 2.0 + np.array([0.1, -0.2, 0.3])
    w = np.full(32, 1.0, np.float32)
    for rmax, want in ((1.4, 1.4 * 1023 / 1024), (4.0, 2.0)):
        P = OracleParams(walks_per_sample=1, eps=1e-4, rmax=rmax)
        _, balls = orc.run_walks(P, False, weight=w, pos=pos)
        assert np.abs(balls[:, 0] - want).max() <= rmax / 1024 + 1e-4
        c = balls[:, 1:4]
        n = (pos - np.array([0.1, -0.2, 0.3])) / 2.0
        assert np.abs(c - (pos - balls[:, :1] * n)).max() < 1e-12


def test_tangent_ball_cube_face_closed_form():
    """Unit cube: r_max = 1/2.  At distance a from a (90 degree) edge, well away from
    the other edges, the largest tangent ball has radius min(a, r_max)."""
    v, f = box((1, 1, 1), (1, 1, 1))
    orc = Oracle(mesh_geom(v, f))
    assert orc.rmax() == 0.5
    # face +x is made of two triangles; pick points by brute force through bary of face 0
    fx = [k for k in range(len(f)) if np.allclose(v[f[k]][:, 0], 0.5)]
    k = fx[0]
    tv = v[f[k]].astype(np.float64)
    rng = np.random.default_rng(0)
    bary = rng.dirichlet(np.ones(3), 200)
    p = bary @ tv
    a = 0.5 - np.abs(p[:, 1:]).max(1)                      # distance to the nearest edge of the face
    P = OracleParams(walks_per_sample=1, eps=1e-6)
    _, balls = orc.run_walks(P, False, tri=np.full(200, k), bary=bary, weight=np.ones(200))
    assert np.abs(balls[:, 0] - np.minimum(a, 0.5)).max() <= 0.5 / 1024 + 1e-6


def test_tangent_ball_exterior_offcentre_sphere():
    """Kelvin image of a sphere (centre c0, radius R, origin inside) is a sphere; the
    normal n* of Eq. 54 must be its outward normal at s*, and every admissible
    tangent ball fits, so r = hi * 1023/1024 with hi = min(r_max, 0.45 |s*|^2 / (s*.n*))."""
    c0, R = np.array([0.3, 0.0, 0.0]), 1.0
    orc = Oracle(sphere_geom(c0, R))
    pos = fibonacci_sphere(64) * R + c0
    P = OracleParams(walks_per_sample=1, eps=1e-6, rmax=10.0, Rmax_norm=1.3)
    _, balls = orc.run_walks(P, True, weight=np.ones(64, np.float32), pos=pos)
    sstar = pos / (pos ** 2).sum(1, keepdims=True)
    den = R * R - c0 @ c0
    cstar_img, r_img = -c0 / den, R / den                  # inverted sphere
    n_true = (sstar - cstar_img) / r_img
    r, c = balls[:, 0], balls[:, 1:4]
    nstar = (sstar - c) / r[:, None]
    assert np.abs(nstar - n_true).max() < 1e-9
    assert np.abs(balls[:, 4] - np.linalg.norm(sstar, axis=1)).max() < 1e-12
    hi = 0.45 * (sstar ** 2).sum(1) / np.einsum("ij,ij->i", sstar, n_true)
    assert np.allclose(r, hi * 1023 / 1024, rtol=1e-12)
    assert (np.linalg.norm(c, axis=1) > r).all()           # the ball does not contain 0


# --------------------------------------------------------------------------
# walk on spheres: exit points follow harmonic measure (Eq. 5)
# --------------------------------------------------------------------------
def _assert_mean_zero(x, nsig=4.5):
    x = np.asarray(x, np.float64)
    se = x.std(ddof=1) / np.sqrt(len(x))
    assert abs(x.mean()) <= nsig * se + 1e-4, (x.mean(), se)


def test_wos_interior_harmonic_functions_sphere_and_mesh():
    # analytic sphere: E[h(t)] = h(z) for harmonic h
    orc = Oracle(sphere_geom((0, 0, 0), 1.0))
    pos = fibonacci_sphere(200)
    P = OracleParams(seed=5, walks_per_sample=64, eps=1e-5, rmax=0.5, importance_sample=False)
    rec, _ = orc.run_walks(P, False, weight=np.ones(200, np.float32), pos=pos)
    ok = rec["steps"] >= 0
    t, z = rec["t"][ok], rec["z"][ok]
    assert (np.abs(np.linalg.norm(t, axis=1) - 1) < 1e-12).all()
    assert rec["steps"][ok].mean() > 3
    pole = np.array([0.4, -1.1, 0.9])                      # outside the ball
    for h in (lambda x: x[:, 0], lambda x: x[:, 2], lambda x: x[:, 0] ** 2 - x[:, 1] ** 2,
              lambda x: x[:, 0] * x[:, 1] * x[:, 2], lambda x: 1 / np.linalg.norm(x - pole, axis=1)):
        _assert_mean_zero(h(t) - h(z))
    # mesh (cube): coordinates are harmonic, E[t] = z
    v, f = box((1, 1, 1), (2, 2, 2))
    orc = Oracle(mesh_geom(v, f))
    smp = uniform_samples(v, f, 300, seed=1)
    P = OracleParams(seed=6, walks_per_sample=32, eps=1e-4, importance_sample=False)
    rec, _ = orc.run_walks(P, False, smp["tri"], smp["bary"], smp["weight"])
    ok = rec["steps"] >= 0
    for k in range(3):
        _assert_mean_zero(rec["t"][ok][:, k] - rec["z"][ok][:, k])
    # exit points are on the surface, on the reported face
    tri = f[rec["tri_t"][ok]]
    cp = np.einsum("qk,qkd->qd", rec["bary_t"][ok], v[tri].astype(np.float64))
    assert np.abs(cp - rec["t"][ok]).max() < 1e-12


@pytest.mark.parametrize("origin", [(0.0, 0.0, 0.0), (0.3, 0.1, -0.2)])
def test_wos_kelvin_harmonic_measure(origin):
    """u(x) = 1/|x - p| (p inside the solid) is harmonic outside and decays, so
    kappa[u](y) = |x| u(x) is harmonic in the inverted domain (Eq. 55): its mean
    over the exit points of walks from z* equals its value at z*; from y = 0
    (killing walks) it equals lim |x| u(x) = 1, and E|t0 - o| is the capacity R."""
    o = np.array(origin)
    R = 1.2
    orc = Oracle(sphere_geom((0, 0, 0), R))
    pos = fibonacci_sphere(150) * R
    P = OracleParams(seed=9, walks_per_sample=64, eps=1e-6, rmax=10.0, importance_sample=False,
                     origin=origin, Rmax_norm=R + np.linalg.norm(o),
                     include_killing=True, n_kill_walks=20000)
    rec, _ = orc.run_walks(P, True, weight=np.ones(150, np.float32), pos=pos)
    ok = rec["steps"] >= 0
    assert ok.all()
    jump, kill = rec[rec["sample"] >= 0], rec[rec["sample"] < 0]
    p = o + np.array([0.2, -0.3, 0.1])

    def kelvin_u(y_or_t, is_kelvin):
        if is_kelvin:
            xt = y_or_t / (y_or_t ** 2).sum(1, keepdims=True)          # x - o
        else:
            xt = y_or_t - o
        return np.linalg.norm(xt, axis=1) / np.linalg.norm(xt + o - p, axis=1)

    _assert_mean_zero(kelvin_u(jump["t"], False) - kelvin_u(jump["z"], True))
    _assert_mean_zero(kelvin_u(kill["t"], False) - 1.0)
    _assert_mean_zero(np.linalg.norm(kill["t"] - o, axis=1) - R)
    assert np.abs(np.linalg.norm(rec["t"], axis=1) - R).max() < 1e-9


# --------------------------------------------------------------------------
# analytic ball: Steklov spectra l (interior) and l + 1 (exterior)
# --------------------------------------------------------------------------
def _cap_spectrum(l, theta0_deg):
    """Expectation of the estimator on the unit ball when the tangent ball is the
    whole ball (Funk-Hecke applied to Eq. 20 with J of Eq. 23 outside the cap)."""
    t0 = np.deg2rad(theta0_deg)
    f = lambda th: (1 - eval_legendre(l, np.cos(th))) * np.cos(th / 2) / (4 * np.sin(th / 2) ** 2)
    return quad(f, t0, np.pi, limit=200)[0]


def _galerkin_from_records(rec, pos_s, centre):
    """S = sum_w weight (Y(s) - Y(t)) (Y(s) - Y(t))^T, killing: weight Y(t) Y(t)^T."""
    jump, kill = rec[rec["sample"] >= 0], rec[rec["sample"] < 0]
    jump = jump[jump["steps"] >= 0]
    Ys = real_sph_harm(pos_s - centre)[jump["sample"]]
    Yt = real_sph_harm(jump["t"] - centre)
    d = Ys - Yt
    S = (d * jump["weight"][:, None]).T @ d
    Sk = np.zeros_like(S)
    if len(kill):
        Yk = real_sph_harm(kill["t"] - centre)
        Sk = (Yk * kill["weight"][:, None]).T @ Yk
    return S, Sk


def test_interior_unit_ball_whole_ball_matches_cap_quadrature():
    n_s, W = 4000, 64
    pos = fibonacci_sphere(n_s)
    orc = Oracle(sphere_geom((0, 0, 0), 1.0))
    for imp in (True, False):
        P = OracleParams(seed=1, walks_per_sample=W, eps=1e-2, rmax=1.0 * 1024 / 1023,
                         importance_sample=imp, cap_half_angle_deg=2.5)
        rec, balls = orc.run_walks(P, False, weight=np.full(n_s, 4 * np.pi / n_s, np.float32), pos=pos)
        assert np.allclose(balls[:, 0], 1.0, atol=1e-12)
        assert (rec["steps"] == 0).all()
        S, _ = _galerkin_from_records(rec, pos, np.zeros(3))
        want = np.array([_cap_spectrum(l, 2.5) for l in DEGREES])
        tol = 0.03 if imp else 0.15
        assert np.abs(np.diag(S) - want).max() < tol, (np.diag(S), want)
        off = S - np.diag(np.diag(S))
        assert np.abs(off).max() < tol


def test_cap_quadrature_tends_to_l():
    for l in range(0, 5):
        assert abs(_cap_spectrum(l, 1e-3) - l) < 1e-3
    assert abs(_cap_spectrum(1, 2.5) - (1 - np.sin(np.deg2rad(1.25)))) < 1e-9


def test_interior_unit_ball_half_radius_walks_give_l():
    """Tangent balls of radius 1/2: now the walks matter.  Small cap, so the
    spectrum is l minus about (l+1) sin(theta0/2)."""
    n_s, W = 6000, 64
    pos = fibonacci_sphere(n_s)
    orc = Oracle(sphere_geom((0, 0, 0), 1.0))
    P = OracleParams(seed=2, walks_per_sample=W, eps=1e-5, rmax=0.5 * 1024 / 1023, cap_half_angle_deg=0.5)
    rec, balls = orc.run_walks(P, False, weight=np.full(n_s, 4 * np.pi / n_s, np.float32), pos=pos)
    assert np.allclose(balls[:, 0], 0.5, atol=1e-9)
    S, _ = _galerkin_from_records(rec, pos, np.zeros(3))
    lam = np.diag(S)
    assert abs(lam[0]) < 1e-12                                        # constants are annihilated
    for k in range(1, len(DEGREES)):
        l = DEGREES[k]
        assert abs(lam[k] - l) < 0.06 * l + 0.02, (l, lam[k])
    off = S - np.diag(lam)
    assert np.abs(off).max() < 0.12


@pytest.mark.parametrize("origin,R", [((0.0, 0.0, 0.0), 1.0), ((0.3, 0.0, 0.0), 1.0), ((0.0, 0.2, 0.1), 2.0)])
def test_exterior_sphere_jump_l_killing_one(origin, R):
    """Exterior Steklov eigenvalues of a sphere are (l+1)/R: jump part l/R
    (Eq. 30 weights |s*|^3/|t*|), killing part K = 1/R (Eq. 31), also when the
    Kelvin origin is off-centre so that both factors are non-trivial."""
    n_s, W = 6000, 64
    o = np.array(origin)
    pos = fibonacci_sphere(n_s) * R
    orc = Oracle(sphere_geom((0, 0, 0), R))
    P = OracleParams(seed=3, walks_per_sample=W, eps=1e-5 / R, rmax=10.0, cap_half_angle_deg=0.5,
                     origin=origin, Rmax_norm=R + np.linalg.norm(o),
                     include_killing=True, n_kill_walks=n_s * W)
    rec, _ = orc.run_walks(P, True, weight=np.full(n_s, 4 * np.pi * R * R / n_s, np.float32), pos=pos)
    assert (rec["steps"] >= 0).all()
    S, Sk = _galerkin_from_records(rec, pos, np.zeros(3))
    # Y is orthonormal on the UNIT sphere: int_{|x|=R} Y_i Y_j = R^2 delta_ij
    lam_jump, lam_kill = np.diag(S) / R ** 2, np.diag(Sk) / R ** 2
    for k, l in enumerate(DEGREES):
        assert abs(lam_jump[k] - l / R) < (0.07 * l + 0.03) / R, ("jump", l, lam_jump[k])
        assert abs(lam_kill[k] - 1 / R) < 0.06 / R, ("kill", l, lam_kill[k])
    assert np.abs(S - np.diag(np.diag(S))).max() / R ** 2 < 0.2 / R
    assert np.abs(Sk - np.diag(np.diag(Sk))).max() / R ** 2 < 0.06 / R
    # capacity: 1^T S_kill 1 = 4 pi E|t0| = 4 pi R
    kill = rec[rec["sample"] < 0]
    assert abs(kill["weight"].sum() - 4 * np.pi * R) < 0.02 * 4 * np.pi * R


# --------------------------------------------------------------------------
# meshes: structural invariants of Alg. 2 / Eq. 32 and sphere multiplicities
# --------------------------------------------------------------------------
@pytest.fixture(scope="module")
def ico2_interior():
    v, f = icosphere(2)
    orc = Oracle(mesh_geom(v, f))
    smp = vertex_cell_samples(v, f, 8, seed=0)
    P = OracleParams(seed=0, walks_per_sample=128, eps=1e-3)
    out = orc.estimate_dtn(P, False, smp["tri"], smp["bary"], smp["weight"], want_var=True)
    return v, f, orc, smp, out


def test_config0_interior_invariants_and_multiplicities(ico2_interior):
    v, f, orc, smp, out = ico2_interior
    S = out["S"]
    assert np.abs(S - S.T).max() <= 1e-15 * np.abs(S).max()            # symmetric by construction
    assert np.linalg.eigvalsh(S).min() >= -1e-12 * np.abs(S).max()     # PSD for any N
    assert np.abs(S.sum(1)).max() <= 1e-6 * np.abs(S).max()            # constants annihilated (385)
    lam = steklov_eigs(S, orc.mass_matrix(), 16)
    assert abs(lam[0]) < 1e-6
    groups = [lam[1:4], lam[4:9], lam[9:16]]
    for l, g in zip((1, 2, 3), groups):
        assert abs(g.mean() - l) < 0.12 * l                            # biased low by cap and eps
        assert g.max() - g.min() < 0.12 * l + 0.05      # MC spread inside a multiplet
    assert groups[1].min() - groups[0].max() > 0.5 and groups[2].min() - groups[1].max() > 0.4
    rec = out["records"]
    assert (rec["steps"] >= 0).all() and 3.0 < rec["steps"].mean() < 5.0
    assert 0.45 < (rec["steps"] == 0).mean() < 0.6


def test_interior_scales_inversely_with_size(ico2_interior):
    v, f, orc, smp, out = ico2_interior
    v2 = (v.astype(np.float64) * 2.0).astype(np.float32)               # exact in fp32
    orc2 = Oracle(mesh_geom(v2, f))
    P2 = OracleParams(seed=0, walks_per_sample=128, eps=2e-3)
    out2 = orc2.estimate_dtn(P2, False, smp["tri"], smp["bary"], smp["weight"] * 4.0)
    assert np.allclose(out2["S"], 2.0 * out["S"], rtol=1e-9, atol=1e-12)
    lam = steklov_eigs(out["S"], orc.mass_matrix(), 9)
    lam2 = steklov_eigs(out2["S"], orc2.mass_matrix(), 9)
    assert np.allclose(lam2[1:], lam[1:] / 2.0, rtol=1e-6)


def test_variance_is_order_one_over_n():
    v, f = icosphere(1)
    orc = Oracle(mesh_geom(v, f))
    tot = []
    for W in (32, 128):
        smp = vertex_cell_samples(v, f, 16, seed=1)
        P = OracleParams(seed=4, walks_per_sample=W, eps=1e-3)
        out = orc.estimate_dtn(P, False, smp["tri"], smp["bary"], smp["weight"], want_var=True)
        tot.append(out["var"].sum())
    assert 3.0 < tot[0] / tot[1] < 5.3                                 # 4x the walks, 1/4 the variance
    # the variance estimate is honest: two seeds differ by about sqrt(2) sigma
    smp = vertex_cell_samples(v, f, 16, seed=1)
    outs = [orc.estimate_dtn(OracleParams(seed=s, walks_per_sample=128, eps=1e-3), False,
                             smp["tri"], smp["bary"], smp["weight"], want_var=True) for s in (11, 12)]
    sig = np.sqrt(outs[0]["var"] + outs[1]["var"])
    m = sig > 0
    zscore = (outs[0]["S"] - outs[1]["S"])[m] / sig[m]
    assert 0.8 < zscore.std() < 1.25
    assert (np.abs(zscore) > 4).mean() < 2e-3


def test_exterior_mesh_sphere_l_plus_one_and_killing_flag():
    v, f = icosphere(2)
    orc = Oracle(mesh_geom(v, f))
    smp = vertex_cell_samples(v, f, 8, seed=0)
    M = orc.mass_matrix()
    base = dict(seed=0, walks_per_sample=128, eps=1e-3, origin=(0.1, 0.0, 0.05))
    off = orc.estimate_dtn(OracleParams(**base), True, smp["tri"], smp["bary"], smp["weight"])
    on = orc.estimate_dtn(OracleParams(**base, include_killing=True, n_kill_walks=len(smp["tri"]) * 128),
                          True, smp["tri"], smp["bary"], smp["weight"])
    for out in (off, on):
        S = out["S"]
        assert np.abs(S - S.T).max() <= 1e-15 * np.abs(S).max()
        assert np.linalg.eigvalsh(S).min() >= -1e-12 * np.abs(S).max()
    assert np.abs(off["S"].sum(1)).max() <= 1e-6 * np.abs(off["S"]).max()      # footnote at PAPER.md:385
    lam_off = steklov_eigs(off["S"], M, 9)
    lam_on = steklov_eigs(on["S"], M, 9)
    assert abs(lam_off[0]) < 1e-6
    assert abs(lam_off[1:4].mean() - 1) < 0.12 and abs(lam_off[4:9].mean() - 2) < 0.25
    assert abs(lam_on[0] - 1) < 0.06                                            # l + 1 with l = 0
    assert abs(lam_on[1:4].mean() - 2) < 0.15 and abs(lam_on[4:9].mean() - 3) < 0.3
    kill = on["records"][on["records"]["sample"] < 0]
    cap = kill["weight"].sum() / (4 * np.pi)
    assert 0.95 < cap < 1.0                                                     # polyhedron inside the unit ball


def test_interior_blocks_vanish_and_exterior_couples_with_decay():
    """the interior operator does not couple disjoint solids, the
    exterior one does, less so as they move apart.  Also the capacity of two unit
    spheres at centre distance 2.5 from the classical image series."""
    norms = []
    for dist in (2.5, 4.0):
        parts = [icosphere(1, 1.0, (-dist / 2, 0, 0)), icosphere(1, 1.0, (dist / 2, 0, 0))]
        v, f, vid, fid = merge_meshes(parts)
        orc = Oracle(mesh_geom(v, f))
        smp = vertex_cell_samples(v, f, 4, seed=2)
        A, B = vid == 0, vid == 1
        if dist == 2.5:
            Si = orc.estimate_dtn(OracleParams(seed=1, walks_per_sample=32, eps=1e-3), False,
                                  smp["tri"], smp["bary"], smp["weight"])["S"]
            assert np.abs(Si[np.ix_(A, B)]).max() == 0.0
        P = OracleParams(seed=1, walks_per_sample=256, eps=1e-3, origin=(-dist / 2, 0, 0),
                         include_killing=(dist == 2.5), n_kill_walks=40000)
        out = orc.estimate_dtn(P, True, smp["tri"], smp["bary"], smp["weight"])
        Se = out["S"]
        norms.append(np.linalg.norm(Se[np.ix_(A, B)]))
        if dist == 2.5:
            kill = out["records"][out["records"]["sample"] < 0]
            cap = kill["weight"].sum() / (4 * np.pi)
            beta = np.arccosh(dist / 2.0)
            series = 2 * np.sinh(beta) * sum((-1) ** (n + 1) / np.sinh(n * beta) for n in range(1, 200))
            assert abs(series - 1.4553) < 1e-3
            assert 0.90 * series < cap < 1.01 * series          # level-1 polyhedra are a bit smaller
    assert norms[0] > 0 and norms[1] > 0 and norms[1] < 0.7 * norms[0]


def test_subset_entry_reproduces_the_full_run():
    """orc_run_walks_subset (sampled outputs for full-size GPU parity) must return exactly the
    records of the full run: same Philox counters (index in the full arrays), same arithmetic."""
    from synth import icosphere, vertex_cell_samples
    v, f = icosphere(1)
    smp = vertex_cell_samples(v, f, 3, seed=5)
    orc = Oracle(mesh_geom(v, f))
    for ext in (False, True):
        p = OracleParams(seed=9, walks_per_sample=6, eps=1e-3, include_killing=ext, n_kill_walks=40 if ext else 0,
                         origin=(0.1, 0.0, -0.05))
        full, _ = orc.run_walks(p, ext, smp["tri"], smp["bary"], smp["weight"])
        ids = np.array([0, 7, 31, len(smp["weight"]) - 1])
        sub = orc.run_walks_subset(p, ext, smp["tri"], smp["bary"], smp["weight"], ids, 4, n_kill_first=10)
        for k, i in enumerate(ids):
            for w in range(4):
                a, b = full[i * 6 + w], sub[k * 4 + w]
                assert a.tobytes() == b.tobytes()
        if ext:
            n_main = len(smp["weight"]) * 6
            assert full[n_main:n_main + 10].tobytes() == sub[len(ids) * 4:].tobytes()


def test_escape_rule_r10b():
    """[R10b] an interior walker whose jump radius exceeds the AABB diagonal is outside the box: cut (-3).
    Correctly oriented closed mesh: never happens.  Normals flipped: the tangent ball sits outside the
    solid; the walkers that leave for good are cut long before max_steps, the others land."""
    from synth import icosphere, vertex_cell_samples
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 1, seed=0)
    orc = Oracle(mesh_geom(v, f))
    p = OracleParams(seed=1, walks_per_sample=8, eps=1e-3, max_steps=4096, rmax=0.5)
    rec, _ = orc.run_walks(p, False, smp["tri"], smp["bary"], smp["weight"])
    assert (rec["steps"] >= 0).all()
    vv = v[f[smp["tri"]]].astype(np.float64)
    nrm = np.cross(vv[:, 1] - vv[:, 0], vv[:, 2] - vv[:, 0])
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    rec, _ = orc.run_walks(p, False, smp["tri"], smp["bary"], smp["weight"], normal=-nrm.astype(np.float32))
    st = rec["steps"]
    assert (st == -1).sum() == 0                       # nobody needs 4096 jumps: escapes are detected
    assert 0.005 < (st == -3).mean() < 0.5             # starts hug the surface (importance sampling): most return, some leave for good
    assert (rec["weight"][st == -3] == 0).all() and (rec["tri_t"][st == -3] == -1).all()


def test_inside_rule_r10c():
    """[R10c] exterior twin of R10b: a walker whose empty ball holds the inversion centre (D > |x - o|) is inside
    the solid: cut (-3).  Closed, outward-oriented mesh: never fires, whatever the centre.  Normals flipped: the
    tangent ball sits inside the solid; every walk either lands on the surface or is cut, long before max_steps
    (in Kelvin coordinates an uncut walker would double |y| per jump), and a cut walker was indeed inside."""
    from synth import icosphere, vertex_cell_samples
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 1, seed=0)
    orc = Oracle(mesh_geom(v, f))
    for origin in [(0.0, 0.0, 0.0), (0.3, -0.2, 0.4)]:
        p = OracleParams(seed=1, walks_per_sample=8, eps=1e-3, max_steps=4096, origin=origin, include_killing=True, n_kill_walks=64)
        rec, _ = orc.run_walks(p, True, smp["tri"], smp["bary"], smp["weight"])
        assert (rec["steps"] >= 0).all()
    vv = v[f[smp["tri"]]].astype(np.float64)
    nrm = np.cross(vv[:, 1] - vv[:, 0], vv[:, 2] - vv[:, 0])
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    p = OracleParams(seed=1, walks_per_sample=8, eps=1e-3, max_steps=4096, origin=(0.3, -0.2, 0.4))
    rec, _ = orc.run_walks(p, True, smp["tri"], smp["bary"], smp["weight"], normal=-nrm.astype(np.float32))
    st = rec["steps"]
    assert (st == -1).sum() == 0 and (st != -2).all()
    assert 0.005 < (st == -3).mean() < 0.9
    assert (rec["weight"][st == -3] == 0).all() and (rec["tri_t"][st == -3] == -1).all()
    # the walks of these samples start inside the unit sphere: Kelvin start z, physical start o + z / |z|^2
    z = rec["z"][st != -2]
    x0 = np.asarray(p.origin) + z / (z ** 2).sum(1, keepdims=True)
    assert (np.linalg.norm(x0, axis=1) < 1.0).all()


# --------------------------------------------------------------------------
# Alg. 1, the naive finite-difference estimator (Eq. 13-16)
# --------------------------------------------------------------------------
def test_naive_estimator_unit_ball_finite_difference_spectrum():
    """On the unit ball the harmonic extension of Y_l is r^l Y_l, so Eq. 14 gives exactly
    (1 - (1 - eps)^l) / eps for degree l (l - l(l-1) eps / 2 + ...): a closed form that pins the start point
    x = s - eps n, the weight |dOmega| / (N eps) and the sign of b_s (b_s - b_t)^T."""
    n_s, W, inset = 4000, 64, 0.05
    pos = fibonacci_sphere(n_s)
    orc = Oracle(sphere_geom((0, 0, 0), 1.0))
    P = OracleParams(seed=4, walks_per_sample=W, eps=1e-4, estimator=1, inset=inset)
    rec, _ = orc.run_walks(P, False, weight=np.full(n_s, 4 * np.pi / n_s, np.float32), pos=pos)
    assert (rec["steps"] >= 1).all()                                     # the inset point is outside the shell
    assert np.allclose(np.linalg.norm(rec["z"], axis=1), 1.0 - inset, atol=1e-12)
    assert np.allclose(rec["weight"], 4 * np.pi / n_s / W / inset, rtol=1e-6)
    Ys = real_sph_harm(pos)[rec["sample"]]
    Yt = real_sph_harm(rec["t"])
    S = (Ys * rec["weight"][:, None]).T @ (Ys - Yt)
    want = np.array([(1 - (1 - inset) ** l) / inset for l in DEGREES])
    assert abs(S[0, 0]) < 1e-9
    assert np.abs(np.diag(S) - want).max() < 0.08, (np.diag(S), want)
    assert np.abs(S - np.diag(np.diag(S))).max() < 0.12


def test_naive_estimator_on_mesh_is_symmetrised_not_psd_and_noisier():
    """PAPER.md:163 (last line) and the two deficiencies listed after Eq. 16: the symmetrised naive estimate
    is symmetric, but PSD only in expectation, and at equal walk count its entries are
    noisier than those of Alg. 2 (Fig. 12's ordering)."""
    from synth import icosphere, vertex_cell_samples
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 4, seed=0)
    orc = Oracle(mesh_geom(v, f))
    naive = orc.estimate_dtn(OracleParams(seed=3, walks_per_sample=32, eps=1e-4, estimator=1, inset=0.02), False,
                             smp["tri"], smp["bary"], smp["weight"], want_var=True)
    jump = orc.estimate_dtn(OracleParams(seed=3, walks_per_sample=32, eps=1e-4), False,
                            smp["tri"], smp["bary"], smp["weight"], want_var=True)
    Sn, Sj = naive["S"], jump["S"]
    assert np.abs(Sn - Sn.T).max() < 1e-15 * np.abs(Sn).max() + 1e-18
    # b_s d^T annihilates constants on the right only (d sums to 0); after symmetrisation the row sums are
    # (1/2) sum_w w d, zero in expectation: the total over the whole matrix is exactly 0
    assert abs(Sn.sum()) < 1e-6 * np.abs(Sn).sum()                       # fp32 barycentrics sum to 1 within 1e-7
    assert np.linalg.eigvalsh(Sn).min() < -1e-3 * np.abs(Sn).max()       # not PSD at finite N
    assert np.linalg.eigvalsh(Sj).min() > -1e-12 * np.abs(Sj).max()      # Alg. 2 is, by construction
    # "the variance blows up as eps is decreased to reduce bias" (deficiency 2): ~1/eps, and above Alg. 2's
    fine = orc.estimate_dtn(OracleParams(seed=3, walks_per_sample=32, eps=1e-5, estimator=1, inset=0.002), False,
                            smp["tri"], smp["bary"], smp["weight"], want_var=True)
    assert fine["var"].mean() > 4.0 * naive["var"].mean()
    assert fine["var"].mean() > 2.0 * jump["var"].mean()
    # still the same operator in expectation: the coordinate functions are the l = 1 harmonics, for which the
    # finite difference is exact on a ball ((1 - (1 - eps)) / eps = 1); Rayleigh quotients, not eigenvalues (not PSD)
    M = orc.mass_matrix()
    for k in range(3):
        g = v[:, k].astype(np.float64)
        assert abs(g @ Sn @ g / (g @ M @ g) - 1.0) < 0.1


# --------------------------------------------------------------------------
# antithetic sampling on the tangent ball ("antithetical sampling on each tangent ball"; reading R7:
# walks 2j and 2j+1 share the INIT draw of counter walk = j and start at azimuths phi and phi + pi; their STEP
# streams stay those of their own walk index)
# --------------------------------------------------------------------------
def _antithetic_setup(W=32, n_s=300, r=0.5, seed=11, eps=1e-3):
    pos = fibonacci_sphere(n_s)
    orc = Oracle(sphere_geom((0, 0, 0), 1.0))
    w = np.full(n_s, 4 * np.pi / n_s, np.float32)
    kw = dict(seed=seed, walks_per_sample=W, eps=eps, rmax=r * 1024 / 1023, cap_half_angle_deg=2.5)
    rec_a, balls = orc.run_walks(OracleParams(antithetic=True, **kw), False, weight=w, pos=pos)
    rec_n, _ = orc.run_walks(OracleParams(antithetic=False, **kw), False, weight=w, pos=pos)
    return pos, balls, rec_a.reshape(n_s, W), rec_n.reshape(n_s, W)


def test_antithetic_partners_are_mirror_images_about_the_pole_axis():
    """The partners' start points have the same polar angle and opposite tangential parts:
    z_{2j} + z_{2j+1} - 2 (c + r cos(theta) n) = 0, (z - c).n equal, |z - c| = r, equal weights; the even partner
    is the start point the plain run gives walk j (shared INIT draw, no shift)."""
    pos, balls, ra, rn = _antithetic_setup()
    r, c = balls[:, 0], balls[:, 1:4]
    n = (pos - c) / r[:, None]                                    # pole: from the centre to the tangent point
    assert np.allclose(np.linalg.norm(n, axis=1), 1.0, atol=1e-12)
    a = ra["z"][:, 0::2] - c[:, None, :]
    b = ra["z"][:, 1::2] - c[:, None, :]
    an = np.einsum("swk,sk->sw", a, n)
    bn = np.einsum("swk,sk->sw", b, n)
    assert np.abs(an - bn).max() < 1e-12
    assert np.abs(a + b - 2 * an[..., None] * n[:, None, :]).max() < 1e-12          # the mirror identity
    assert np.abs(np.linalg.norm(a, axis=2) - r[:, None]).max() < 1e-12
    at = a - an[..., None] * n[:, None, :]
    assert np.linalg.norm(at, axis=2).min() > 1e-6                # outside the cap: the two points are distinct
    assert np.array_equal(ra["weight"][:, 0::2], ra["weight"][:, 1::2])
    W = ra.shape[1]
    assert np.abs(ra["z"][:, 0::2] - rn["z"][:, :W // 2]).max() == 0.0               # even partner = plain walk j's start


def test_antithetic_partners_keep_their_own_step_streams():
    """Each partner's jumps are drawn from Philox(seed; sample, ITS OWN walk index, step, STEP): re-walking from the
    recorded start point on the analytic unit ball (distance 1 - |x|) with those counters, through the generator that
    is pinned against cuRAND, lands on the recorded exit point.  Sharing the stream between partners (walk >> 1)
    would not."""
    from oracle import philox4x32_10, u01
    seed, eps = 11, 1e-3
    pos, balls, ra, rn = _antithetic_setup(W=8, n_s=40, seed=seed, eps=eps)
    shared_would_differ = 0
    for i in range(ra.shape[0]):
        for w in range(ra.shape[1]):
            for stream in (w, w >> 1):
                x = ra["z"][i, w].copy()
                k = 0
                while True:
                    d = 1.0 - np.linalg.norm(x)
                    if d < eps:
                        break
                    k += 1
                    words = philox4x32_10((i, stream, k, 2), (seed & 0xFFFFFFFF, seed >> 32))
                    ct = 1.0 - 2.0 * u01(words[0])
                    st = np.sqrt(max(0.0, 1.0 - ct * ct))
                    phi = 2.0 * np.pi * u01(words[1])
                    x += d * np.array([st * np.cos(phi), st * np.sin(phi), ct])
                t = x / np.linalg.norm(x)
                if stream == w:
                    assert k == ra["steps"][i, w]
                    assert np.abs(t - ra["t"][i, w]).max() < 1e-9
                elif w >= 2 and k > 0:                            # walks 0, 1: w >> 1 == 0 is walk 0's own stream
                    shared_would_differ += int(np.abs(t - ra["t"][i, w]).max() > 1e-6)
    assert shared_would_differ > 50                               # the check above has teeth


def test_interior_unit_ball_whole_ball_cap_spectrum_holds_with_antithetic_pairs():
    """Antithetic partners are each distributed as a plain start point, so the expectation is unchanged: the
    whole-ball case (no walk) must still give the cap quadrature (phi + pi/2, or a pair sharing one point, would not
    change this; the mirror identity above pins those)."""
    n_s, W = 8000, 64            # partners share their polar angle, so even functionals (d d^T) see half as many draws
    pos = fibonacci_sphere(n_s)
    orc = Oracle(sphere_geom((0, 0, 0), 1.0))
    P = OracleParams(seed=1, walks_per_sample=W, eps=1e-2, rmax=1.0 * 1024 / 1023, cap_half_angle_deg=2.5, antithetic=True)
    rec, balls = orc.run_walks(P, False, weight=np.full(n_s, 4 * np.pi / n_s, np.float32), pos=pos)
    assert (rec["steps"] == 0).all()
    S, _ = _galerkin_from_records(rec, pos, np.zeros(3))
    want = np.array([_cap_spectrum(l, 2.5) for l in DEGREES])
    assert np.abs(np.diag(S) - want).max() < 0.03, (np.diag(S), want)
    assert np.abs(S - np.diag(np.diag(S))).max() < 0.03


def test_antithetic_pairs_cancel_odd_tangential_moments():
    """What the pairing buys: a functional that is odd in the tangential offset of the start point has a pair sum of
    exactly zero at the start points (here: the tangential part of z - c), and the pair means of first-order
    quantities of the exit points, E[t - s] projected on a tangent direction, have a smaller variance than means over
    independent pairs."""
    pos, balls, ra, rn = _antithetic_setup(W=64, n_s=400, eps=1e-4)
    r, c = balls[:, 0], balls[:, 1:4]
    n = (pos - c) / r[:, None]
    e = np.cross(n, np.array([0.3, -0.5, 0.8]))
    e /= np.linalg.norm(e, axis=1, keepdims=True)                  # a tangent direction per sample
    fa = np.einsum("swk,sk->sw", ra["t"] - pos[:, None, :], e)
    fn = np.einsum("swk,sk->sw", rn["t"] - pos[:, None, :], e)
    var_pairs_anti = (0.5 * (fa[:, 0::2] + fa[:, 1::2])).var()
    var_pairs_plain = (0.5 * (fn[:, 0::2] + fn[:, 1::2])).var()
    assert var_pairs_anti < 0.8 * var_pairs_plain, (var_pairs_anti, var_pairs_plain)


# --------------------------------------------------------------------------
# thin spots named by the round-1 review: r_max of the exterior rule and the AABB diagonal of R10b
# --------------------------------------------------------------------------
def test_aabb_diagonal_and_exterior_rmax_closed_forms():
    import ctypes as C
    v, f = box((1.0, 2.0, 3.0), (2, 2, 2))
    orc = Oracle(mesh_geom(v, f))
    orc.lib.orc_aabb_diagonal.restype = C.c_double
    assert abs(orc.lib.orc_aabb_diagonal(C.byref(orc.geom.c)) - np.sqrt(14.0)) < 1e-6      # half of it would fail
    assert abs(orc.rmax() - 0.5) < 1e-7                                                    # half the shortest side
    # exterior: AABB of the inverted vertices (PAPER.md:642 applied in the inverted domain, R11).  Unit sphere about
    # its centre: kappa fixes the sphere, sides 2, r_max = 1.  About an interior point at distance a from the centre
    # the image is a sphere of radius R / (R^2 - a^2): r_max = that radius (up to the tessellation).
    v, f = icosphere(4)
    orc = Oracle(mesh_geom(v, f))
    assert abs(orc.rmax(True, (0.0, 0.0, 0.0)) - 1.0) < 2e-3
    a = 0.3
    assert abs(orc.rmax(True, (a, 0.0, 0.0)) - 1.0 / (1.0 - a * a)) < 5e-3
    v2, f2 = icosphere(4, radius=2.0)
    assert abs(Oracle(mesh_geom(v2, f2)).rmax(True, (0.0, 0.5, 0.0)) - 2.0 / (4.0 - 0.25)) < 5e-3


def test_exterior_tangent_ball_stays_out_of_a_neighbouring_solid():
    """Readings E2 + R4: the accepted Kelvin ball may poke out of the inverted domain by at most eps/2 IN KELVIN
    COORDINATES.  BASELINE config 2b in small (two unit spheres 2.5 apart, the torus between them, inversion centre =
    centre of the first sphere A, whose image is the unit sphere |y| = 1 with A's inside OUTSIDE it): tangent balls of
    torus samples grow until they meet the image of A, and some of them pass close to 0 = kappa(infinity), where their
    primal image is a huge ball.  Every accepted ball must stay within |y| <= 1 + eps.  An earlier form of the test
    shrank the primal image by the RELATIVE amount eps / 2r, i.e. by eps / (2 (|c*|^2 - r^2)) in primal units, and let
    such balls reach 0.014 into A (found by the full-size GPU test of config 2b: walks started inside A, two of 83 M
    were cut by R10c on both sides)."""
    from synth import torus
    parts = [icosphere(3, 1.0, (-1.25, 0, 0)), icosphere(3, 1.0, (1.25, 0, 0)), torus(1.0, 0.3, 60, 30, axis="x")]
    v, f, vid, fid = merge_meshes(parts)
    orc = Oracle(mesh_geom(v, f))
    origin = (-1.25, 0.0, 0.0)
    tor = np.flatnonzero(fid == 2)
    eps = 1e-3
    P = OracleParams(walks_per_sample=1, eps=eps, origin=origin)
    rec, balls = orc.run_walks(P, True, tor.astype(np.int32), np.full((len(tor), 3), 1 / 3, np.float32), np.ones(len(tor), np.float32))
    r, c = balls[:, 0], balls[:, 1:4]
    ok = r > 0
    assert ok.mean() > 0.95
    near_origin = ok & ((np.linalg.norm(c, axis=1) ** 2 - r ** 2) < 0.05)      # balls whose primal image is large
    assert near_origin.sum() > 20
    pick = np.flatnonzero(near_origin)[:60]
    # points on those Kelvin balls, mapped back to primal space: how deep do they sit inside a solid?
    u = fibonacci_sphere(96)
    y = (c[pick, None, :] + r[pick, None, None] * u[None, :, :]).reshape(-1, 3)
    x = np.asarray(origin) + y / (y ** 2).sum(1, keepdims=True)
    D = orc.closest_points(x.astype(np.float32))["dist"]
    inside = orc.winding_number(x) > 0.5
    rho = np.linalg.norm(x - np.asarray(origin), axis=1)
    # allowed: eps/2 in Kelvin coordinates = (eps/2) rho^2 in primal ones (|kappa(x) - kappa(p)| = |x - p| / (|x||p|))
    depth = np.where(inside, D, 0.0)
    assert inside.sum() < 0.02 * len(x)
    assert (depth <= 0.75 * eps * np.maximum(rho, 1.0) ** 2 + 1e-5).all(), (depth.max(), rho[depth.argmax()])
    reach = np.linalg.norm(c, axis=1) + r
    assert reach[ok].max() > 0.97                                  # some balls are limited by A: they nearly touch its image
