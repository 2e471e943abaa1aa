"""Real orthonormal spherical harmonics on the unit sphere (test helper, textbook
formulas): all of l <= 2 plus the zonal l = 3, 4.  Returns (values [n, 11], degrees)."""
import numpy as np

DEGREES = np.array([0, 1, 1, 1, 2, 2, 2, 2, 2, 3, 4])


def real_sph_harm(p):
    p = np.asarray(p, np.float64)
    p = p / np.linalg.norm(p, axis=1, keepdims=True)
    x, y, z = p[:, 0], p[:, 1], p[:, 2]
    pi = np.pi
    cols = [np.full_like(x, 0.5 / np.sqrt(pi)),
            np.sqrt(3 / (4 * pi)) * x, np.sqrt(3 / (4 * pi)) * y, np.sqrt(3 / (4 * pi)) * z,
            np.sqrt(15 / (4 * pi)) * x * y, np.sqrt(15 / (4 * pi)) * y * z, np.sqrt(15 / (4 * pi)) * x * z,
            np.sqrt(5 / (16 * pi)) * (3 * z * z - 1), np.sqrt(15 / (16 * pi)) * (x * x - y * y),
            np.sqrt(7 / (4 * pi)) * 0.5 * (5 * z ** 3 - 3 * z),
            np.sqrt(9 / (4 * pi)) * 0.125 * (35 * z ** 4 - 30 * z * z + 3)]
    return np.stack(cols, 1)


def fibonacci_sphere(n):
    """n quasi-uniform points on the unit sphere (equal quadrature weight 4 pi / n)."""
    k = np.arange(n) + 0.5
    z = 1 - 2 * k / n
    phi = np.pi * (1 + 5 ** 0.5) * k
    r = np.sqrt(1 - z * z)
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], 1)
