"""Pins for the oracle's Steklov eigen step (S psi = lambda M psi with lumped mass): cases whose
answer is known without the routine -- a diagonal pencil, a hand-worked 2x2 pencil, the graph Laplacian of a cycle
(closed-form cosine spectrum, constants in the null space) -- plus M-orthonormality and residuals."""
import numpy as np

from oracle import steklov_eigpairs, steklov_eigs


def test_diagonal_pencil():
    s = np.array([3.0, 1.0, 8.0, 0.5])
    m = np.array([1.0, 4.0, 2.0, 0.25])
    w, V = steklov_eigpairs(np.diag(s), m, 4)
    order = np.argsort(s / m)
    assert np.allclose(w, (s / m)[order], rtol=1e-13)
    for e, i in enumerate(order):
        expect = np.zeros(4); expect[i] = 1 / np.sqrt(m[i])
        assert np.allclose(np.abs(V[e]), expect, atol=1e-13)


def test_hand_worked_2x2():
    # S = [[2,-1],[-1,2]], M = diag(1,4):  det(S - l M) = 4 l^2 - 10 l + 3  =>  l = (5 -+ sqrt(13)) / 4
    S = np.array([[2.0, -1.0], [-1.0, 2.0]])
    w, V = steklov_eigpairs(S, np.array([1.0, 4.0]), 2)
    assert np.allclose(w, [(5 - np.sqrt(13)) / 4, (5 + np.sqrt(13)) / 4], rtol=1e-14)
    for l, psi in zip(w, V):
        assert np.allclose((2 - l) * psi[0] - psi[1], 0, atol=1e-13)       # first row of (S - l M) psi = 0
    assert np.allclose(steklov_eigs(S, np.diag([1.0, 4.0]), 2), w, rtol=1e-14)


def test_cycle_laplacian_spectrum():
    n = 24
    S = 2 * np.eye(n) - np.roll(np.eye(n), 1, 0) - np.roll(np.eye(n), -1, 0)
    w, V = steklov_eigpairs(S, np.full(n, 0.5), n)
    expect = np.sort(2 * (2 - 2 * np.cos(2 * np.pi * np.arange(n) / n)))      # (2 - 2 cos) / 0.5
    assert np.allclose(w, expect, atol=1e-12)
    assert np.allclose(np.abs(V[0]), np.sqrt(2.0 / n), atol=1e-12)             # constant null vector, M-normalised
    assert np.allclose(V @ np.diag(np.full(n, 0.5)) @ V.T, np.eye(n), atol=1e-12)


def test_residual_and_asymmetric_input_is_symmetrised():
    rng = np.random.default_rng(3)
    A = rng.normal(size=(30, 30))
    S = A @ A.T
    m = rng.uniform(0.2, 3.0, 30)
    noise = rng.normal(size=(30, 30)) * 1e-3
    w, V = steklov_eigpairs(S + noise - noise.T, m, 7)                         # the antisymmetric part must not matter
    for l, psi in zip(w, V):
        assert np.abs(S @ psi - l * m * psi).max() < 1e-10 * np.abs(S).max()
    assert np.allclose((V * m) @ V.T, np.eye(7), atol=1e-12)
