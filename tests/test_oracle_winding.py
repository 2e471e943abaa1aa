"""Pins for the oracle's generalised winding number and the sidedness rule G-R1:
values fixed by topology (closed surfaces: 1 inside, 0 outside, whatever the tessellation), closed-form solid
angles (an octant, a rectangle seen from above its centre), orientation reversal, a hemisphere seen from its
centre, the exclusion of one face, and the recovery of outward normals on a sphere with randomly flipped faces."""
import numpy as np

from oracle import Oracle, mesh_geom
from synth import box, icosphere, merge_meshes, torus


def _orc(v, f):
    return Oracle(mesh_geom(np.asarray(v, np.float32), np.asarray(f, np.int32)))


def test_closed_surfaces_one_inside_zero_outside():
    rng = np.random.default_rng(0)
    v, f = icosphere(2)
    inside = rng.normal(size=(40, 3)); inside *= (0.9 * rng.random(40) ** (1 / 3) / np.linalg.norm(inside, axis=1))[:, None]
    outside = rng.normal(size=(40, 3)); outside *= ((1.05 + 3 * rng.random(40)) / np.linalg.norm(outside, axis=1))[:, None]
    orc = _orc(v, f)
    assert np.abs(orc.winding_number(inside) - 1).max() < 1e-12
    assert np.abs(orc.winding_number(outside)).max() < 1e-12
    # a torus (genus 1) and two disjoint components: still 1 inside the solid, 0 in the hole and outside
    tv, tf = torus(1.0, 0.3, 40, 20, axis="z")[:2]
    w = _orc(tv, tf).winding_number(np.array([[1.0, 0, 0], [0, 0, 0], [0, 0, 2.0], [0.0, -1.0, 0.1]]))
    assert np.allclose(w, [1, 0, 0, 1], atol=1e-12)
    mv, mf = merge_meshes([icosphere(1), icosphere(1, center=(3, 0, 0))])[:2]
    w = _orc(mv, mf).winding_number(np.array([[0.0, 0, 0], [3.0, 0, 0], [1.5, 0, 0]]))
    assert np.allclose(w, [1, 1, 0], atol=1e-12)
    # nested, both outward: 2 in the inner solid (the paper's "nested geometry")
    nv, nf = merge_meshes([icosphere(1), icosphere(1, radius=0.4)])[:2]
    assert np.allclose(_orc(nv, nf).winding_number(np.array([[0.0, 0, 0], [0.7, 0, 0]])), [2, 1], atol=1e-12)


def test_closed_form_solid_angles():
    # the triangle (e1, e2, e3) seen from the origin cuts out one octant: Omega = 4 pi / 8
    v = np.array([[1.0, 0, 0], [0, 1, 0], [0, 0, 1]]); f = np.array([[0, 1, 2]])
    assert abs(_orc(v, f).winding_number(np.zeros((1, 3)))[0] - 1 / 8) < 1e-15
    assert abs(_orc(v, f[:, ::-1]).winding_number(np.zeros((1, 3)))[0] + 1 / 8) < 1e-15      # reversed winding
    # rectangle of half-sides a, b seen from height h above its centre: Omega = 4 atan(a b / (h sqrt(a^2 + b^2 + h^2)))
    a, b, h = 0.75, 1.25, 0.5                     # exactly representable in fp32
    v = np.array([[-a, -b, 0], [a, -b, 0], [a, b, 0], [-a, b, 0]]); f = np.array([[0, 1, 2], [0, 2, 3]])
    want = 4 * np.arctan(a * b / (h * np.sqrt(a * a + b * b + h * h))) / (4 * np.pi)
    w = _orc(v, f).winding_number(np.array([[0, 0, h], [0, 0, -h]]))
    assert abs(w[0] + want) < 1e-14 and abs(w[1] - want) < 1e-14                               # counter-clockwise from +z: +z is outside


def test_open_hemisphere_is_one_half_at_the_centre():
    v, f = icosphere(3)
    keep = (v[f].mean(1)[:, 2] > 0)
    w = _orc(v, f[keep]).winding_number(np.zeros((1, 3)))[0]
    assert abs(w - 0.5) < 0.02                                                                 # the rim is a zig-zag of the equator


def test_exclusion_removes_exactly_one_face():
    v, f = icosphere(1)
    orc = _orc(v, f)
    p = np.array([[0.2, 0.1, -0.3], [1.5, 0.2, 0.1]])
    w_all = orc.winding_number(p)
    w_ex = orc.winding_number(p, exclude=[7, 7])
    single = _orc(v, f[7:8]).winding_number(p)
    assert np.abs(w_all - w_ex - single).max() < 1e-14


def test_sidedness_finds_flipped_faces():
    """G-R1 on a sphere and a box + torus scene with 10 % of the faces reversed: the returned normal points out of
    the solid for every sample; d > 0 exactly on the faces that kept their orientation."""
    rng = np.random.default_rng(3)
    v, f = icosphere(3)
    flip = rng.random(len(f)) < 0.1
    f2 = f.copy(); f2[flip] = f2[flip][:, ::-1]
    tri = rng.integers(0, len(f), 300).astype(np.int32)
    bary = rng.dirichlet([1, 1, 1], 300).astype(np.float32)
    nrm, d = _orc(v, f2).orient_samples(tri, bary, h_scale=1.0)
    s = np.einsum("qk,qkd->qd", bary.astype(np.float64), v[f2[tri]].astype(np.float64))
    assert (np.einsum("qd,qd->q", nrm, s) > 0).all()
    assert ((d > 0) == ~flip[tri]).all()
    # unflipped closed surface: nothing changes, d ~ the jump of a smooth field over 2 h: positive, below 1
    nrm0, d0 = _orc(v, f).orient_samples(tri, bary, h_scale=1.0)
    assert (d0 > 0).all() and (d0 < 1).all()
