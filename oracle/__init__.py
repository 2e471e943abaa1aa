"""CPU oracle for the Monte Carlo DtN estimator -- TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` legs may import this package.  It never imports
`paper_2606_05581_b200` and shares no code with it.  See dtn_oracle.c for the
algorithm (restated from PAPER.md) and for the list of pins.
"""
from .oracle import (Oracle, OracleParams, mesh_geom, sphere_geom, philox4x32_10, u01,
                     closest_point_triangle, closest_point_triangle_alt, inverted_ratio2_triangle,
                     RECORD_DTYPE, steklov_eigs, steklov_eigpairs, PointBasis)

__all__ = ["Oracle", "OracleParams", "mesh_geom", "sphere_geom", "philox4x32_10", "u01",
           "closest_point_triangle", "closest_point_triangle_alt", "inverted_ratio2_triangle", "RECORD_DTYPE",
           "steklov_eigs", "steklov_eigpairs", "PointBasis"]
