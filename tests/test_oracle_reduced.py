"""Pins for the oracle's reduced Ritz-Galerkin accumulation: linearity fixes it
completely -- with phi_k = sum_v Phi[v,k] hat_v the reduced matrix is Phi^T S Phi for the nodal (hat-basis) matrix S
of the same walks, which the C oracle accumulates by a different route (entry by entry from 3-sparse vectors);
Phi = I gives S back; a constant basis function lies in the interior kernel; a basis function supported on one
component only sees that component's block; and sampled spherical harmonics give the sphere spectrum."""
import numpy as np

from oracle import Oracle, OracleParams, mesh_geom
from synth import icosphere, merge_meshes, vertex_cell_samples


def _run(exterior, seed=2, W=16):
    v, f = icosphere(2)
    smp = vertex_cell_samples(v, f, 2, seed=1)
    orc = Oracle(mesh_geom(v, f))
    P = OracleParams(seed=seed, walks_per_sample=W, eps=1e-3, include_killing=exterior, n_kill_walks=4000 if exterior else 0)
    out = orc.estimate_dtn(P, exterior, smp["tri"], smp["bary"], smp["weight"])
    return v, f, smp, orc, out


def test_reduced_is_projection_of_nodal_matrix_interior_and_exterior():
    rng = np.random.default_rng(0)
    for exterior in (False, True):
        v, f, smp, orc, out = _run(exterior)
        Phi = rng.normal(size=(len(v), 7))
        R = orc.accumulate_reduced(out["records"], smp["tri"], smp["bary"], Phi)
        want = Phi.T @ out["S"] @ Phi
        assert np.abs(R - want).max() < 1e-11 * np.abs(want).max()
        assert np.abs(R - R.T).max() < 1e-12 * np.abs(R).max()
        assert np.linalg.eigvalsh(R).min() > -1e-10 * np.abs(R).max()                 # PSD by construction (sum of w d d^T, w > 0)
        I = orc.accumulate_reduced(out["records"], smp["tri"], smp["bary"], np.eye(len(v)))
        assert np.abs(I - out["S"]).max() < 1e-12 * np.abs(out["S"]).max()


def test_constants_are_in_the_interior_kernel_not_the_exterior_one():
    v, f, smp, orc, out = _run(False, W=128)
    Phi = np.concatenate([np.ones((len(v), 1)), v.astype(np.float64)], 1)               # 1, x, y, z
    R = orc.accumulate_reduced(out["records"], smp["tri"], smp["bary"], Phi)
    assert np.abs(R[0]).max() < 1e-7 * np.abs(R).max()                                  # fp32 barycentrics sum to 1 within 6e-8
    # x, y, z restricted to the unit sphere are the degree-1 harmonics: Rayleigh quotient l = 1 (interior)
    v2, f2, smp2, orc2, out2 = _run(True, W=128)
    Re = orc2.accumulate_reduced(out2["records"], smp2["tri"], smp2["bary"], Phi)
    assert Re[0, 0] > 0.5 * 4 * np.pi                                                    # capacity of the unit sphere: 4 pi (l + 1 = 1 for the constant)
    mass = 4 * np.pi / 3                                                                 # int x^2 over the unit sphere
    assert np.all(np.abs(np.diag(R)[1:] / mass - 1.0) < 0.25)
    assert np.all(np.abs(np.diag(Re)[1:] / mass - 2.0) < 0.45)                           # exterior: l + 1 = 2


def test_basis_on_one_component_sees_only_that_component_interior():
    va, fa = icosphere(1)
    v, f = merge_meshes([(va, fa), icosphere(1, center=(3, 0, 0))])[:2]
    smp = vertex_cell_samples(v, f, 2, seed=3)
    orc = Oracle(mesh_geom(v, f))
    out = orc.estimate_dtn(OracleParams(seed=1, walks_per_sample=8, eps=1e-3), False, smp["tri"], smp["bary"], smp["weight"])
    rng = np.random.default_rng(1)
    Phi = np.zeros((len(v), 4)); Phi[:len(va), :2] = rng.normal(size=(len(va), 2)); Phi[len(va):, 2:] = rng.normal(size=(len(v) - len(va), 2))
    R = orc.accumulate_reduced(out["records"], smp["tri"], smp["bary"], Phi)
    assert np.abs(R[:2, 2:]).max() == 0.0                                                # interior walks never leave their component
