"""GPU parity at BASELINE.json's full size, in the launch configuration bench.py times
(configs[1]: icosphere L4, 2562 vertices x 4096 walks per operator as 16 sample points x 256
walks, eps 1e-3, cap 2.5 deg, seed 0).  The brute-force oracle cannot run 10.5M walks, so:
sampled outputs (records of seeded sample points, computed one by one by the oracle with the
same Philox counters) and properties that hold at any size (exact symmetry, bit-identical
rerun, zero row sums, the sphere spectrum l / l+1 with multiplicity 2l+1, capacity)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from bench import make_cfg1                                                      # noqa: E402
from oracle import Oracle, OracleParams, mesh_geom, steklov_eigs              # noqa: E402


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from paper_2606_05581_b200 import api as _api
    _api.lib()
    return _api


@pytest.fixture(scope="module")
def cfg1(api):
    wl = make_cfg1(4, 4096, 16, 0)
    vd = torch.as_tensor(wl["v"]).cuda()
    fd = torch.as_tensor(wl["f"]).cuda()
    bvh = api.build_bvh(vd, fd)
    S = api.Samples.from_arrays(wl["smp"]["tri"], wl["smp"]["bary"], wl["smp"]["weight"])
    orc = Oracle(mesh_geom(wl["v"], wl["f"]))
    return wl, bvh, S, orc


def _sampled_records(api, cfg1, exterior):
    wl, bvh, S, orc = cfg1
    n_walks = wl["n_s"] * wl["W"]
    kw = dict(seed=0, walks_per_sample=wl["W"], eps=1e-3, include_killing=exterior, n_kill_walks=n_walks if exterior else 0)
    rec, steps, st = api.run_walks(bvh, S, api.Params(**kw), exterior, want_stats=True)
    assert st.n_walks == n_walks * (2 if exterior else 1) and st.n_truncated == 0 and st.n_discarded == 0
    rec, steps = rec.cpu().numpy(), steps.cpu().numpy()
    ids = np.sort(np.random.default_rng(1).choice(wl["n_s"], 48, replace=False))
    n_w, n_kill = 8, 256
    orec = orc.run_walks_subset(OracleParams(**kw), exterior, wl["smp"]["tri"], wl["smp"]["bary"], wl["smp"]["weight"],
                                ids, n_w, n_kill_first=n_kill)
    slots = (ids[:, None] * wl["W"] + np.arange(n_w)[None, :]).ravel()
    if exterior:
        slots = np.concatenate([slots, n_walks + np.arange(n_kill)])
    g_steps, g_rec = steps[slots], rec[slots]
    same = g_steps == orec["steps"]
    assert same.mean() >= 0.96, same.mean()
    ok = same & (g_steps >= 0)
    tri_t = g_rec[:, 0].copy().view(np.int32)
    assert (tri_t[ok] == orec["tri_t"][ok]).mean() > 0.97
    v, f = wl["v"], wl["f"]
    bt = np.stack([1 - g_rec[:, 1] - g_rec[:, 2], g_rec[:, 1], g_rec[:, 2]], 1).astype(np.float64)
    t_gpu = np.einsum("qk,qkd->qd", bt[ok], v[f[tri_t[ok]]].astype(np.float64))
    err = np.linalg.norm(t_gpu - orec["t"][ok], axis=1)
    assert np.quantile(err, 0.98) < 2e-4, np.quantile(err, [0.5, 0.98, 1.0])
    rel = np.abs(g_rec[ok, 3] - orec["weight"][ok]) / np.abs(orec["weight"][ok]).max()
    assert np.quantile(rel, 0.98) < 1e-4


def test_config1_interior_full_size(api, cfg1):
    wl, bvh, S, orc = cfg1
    _sampled_records(api, cfg1, False)
    P = api.Params(seed=0, walks_per_sample=wl["W"], eps=1e-3)
    A = api.estimate_dtn_interior(bvh, S, P)
    assert torch.equal(A, api.estimate_dtn_interior(bvh, S, P))                # bit-identical rerun
    assert torch.equal(A, A.T)                                                  # exactly symmetric
    Sg = A.cpu().numpy().astype(np.float64)
    assert np.abs(Sg.sum(1)).max() < 5e-5 * np.abs(Sg).max()                    # annihilates constants
    lam = steklov_eigs(Sg, orc.mass_matrix(), 16)
    assert abs(lam[0]) < 1e-3
    # multiplicities 1, 3, 5, 7; multiplet means sit below l by the cap / eps-shell bias
    for l, sl in ((1, slice(1, 4)), (2, slice(4, 9)), (3, slice(9, 16))):
        m = lam[sl]
        assert 0.88 < m.mean() / l < 1.01, (l, m)
        assert m.max() - m.min() < 0.06 * l, (l, m)
    assert lam[4] - lam[3] > 0.5 and lam[9] - lam[8] > 0.5                      # gaps between multiplets


def test_config1_exterior_full_size(api, cfg1):
    wl, bvh, S, orc = cfg1
    _sampled_records(api, cfg1, True)
    n_walks = wl["n_s"] * wl["W"]
    P = api.Params(seed=0, walks_per_sample=wl["W"], eps=1e-3, include_killing=True, n_kill_walks=n_walks)
    A = api.estimate_dtn_exterior(bvh, S, P)
    assert torch.equal(A, api.estimate_dtn_exterior(bvh, S, P))
    assert torch.equal(A, A.T)
    Sg = A.cpu().numpy().astype(np.float64)
    # jump part annihilates constants, so 1^T S 1 = 4 pi * capacity; unit sphere: capacity 1 (polyhedron: slightly below)
    cap = Sg.sum() / (4 * np.pi)
    assert 0.985 < cap < 1.001, cap
    lam = steklov_eigs(Sg, orc.mass_matrix(), 9)
    assert 0.95 < lam[0] < 1.02, lam[0]                                         # l + 1 with l = 0
    assert 0.9 < lam[1:4].mean() / 2.0 < 1.01 and lam[1:4].max() - lam[1:4].min() < 0.1, lam[1:4]
    assert 0.9 < lam[4:9].mean() / 3.0 < 1.01, lam[4:9]


def test_config1_both_operators_full_size_in_the_configuration_bench_times(api, cfg1):
    """bench.py's step: mcs_estimate_dtn_both with bench.py's parameters (cap 2.5 deg, killing on, seed 0), the two
    walk kernels overlapped.  Bit-identical to the single calls checked above and to itself across reruns."""
    wl, bvh, S, orc = cfg1
    n_walks = wl["n_s"] * wl["W"]
    Pi = api.Params(seed=0, walks_per_sample=wl["W"], eps=1e-3, cap_half_angle_deg=2.5)
    Pe = api.Params(seed=0, walks_per_sample=wl["W"], eps=1e-3, cap_half_angle_deg=2.5, include_killing=True, n_kill_walks=n_walks)
    Ai = api.estimate_dtn_interior(bvh, S, Pi).clone()
    Ae = api.estimate_dtn_exterior(bvh, S, Pe).clone()
    ws = torch.empty(api.workspace_bytes_both(bvh, S, Pi, Pe), dtype=torch.uint8, device="cuda")
    for _ in range(3):
        Bi, Be = api.estimate_dtn_both(bvh, S, Pi, Pe, workspace=ws)
        assert torch.equal(Bi, Ai) and torch.equal(Be, Ae)
    Sg = Bi.cpu().numpy().astype(np.float64)
    assert np.abs(Sg.sum(1)).max() < 5e-5 * np.abs(Sg).max()
    cap = Be.double().sum().item() / (4 * np.pi)
    assert 0.985 < cap < 1.001, cap
