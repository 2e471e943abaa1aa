"""Seeded synthetic input generators (meshes, boundary samples, query sets).

This package serves BOTH the CPU oracle tests and the CUDA path's tests/bench.
It holds none of the method's arithmetic (no closest-point code, no walk, no
estimator weights, no Philox): only geometry construction and sampling of
surface points with numpy's own generators.  Neither `oracle/` nor
`paper_2606_05581_b200/` imports it; only `tests/`, `bench.py` and
`__graft_entry__.py` do.

The paper evaluates on Thingi10k / Objaverse; those are not
available, so these generators stand in for them with the same kinds of shapes
(hundreds to millions of faces, many components, slivers, duplicates, flips).
"""
from .meshes import (icosphere, torus, box, cylinder, merge_meshes, transform,
                     two_spheres_torus_scene, stress_mesh, mesh_area)
from .samples import vertex_cell_samples, uniform_samples, fps_samples
from .queries import near_surface_queries, far_field_queries

__all__ = [
    "icosphere", "torus", "box", "cylinder", "merge_meshes", "transform",
    "two_spheres_torus_scene", "stress_mesh", "mesh_area",
    "vertex_cell_samples", "uniform_samples", "fps_samples",
    "near_surface_queries", "far_field_queries",
]
