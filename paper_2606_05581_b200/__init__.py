"""B200-native (sm_100a, hand-written CUDA) Monte Carlo Dirichlet-to-Neumann
estimator: the walk-on-spheres hot path of arxiv 2606.05581, behind
the C ABI of include/mcdtn.h.  This package is only the thin binding; it never
imports `oracle/` and has no CPU fallback."""
from .api import (steklov_eigs, project_galerkin, project_galerkin_coo, winding_number, orient_samples, CooMatrix, PointBasis, estimate_dtn_coo, knn_weights, Bvh, BvhInfo, McsError, Params, Samples, Stats, accumulate, build_bvh, closest_point,
                  closest_point_bruteforce, estimate_dtn_exterior, estimate_dtn_host, estimate_dtn_interior, launch_count, lib, num_records,
                  philox4x32_10, profile_enable, profile_last, run_walks, sort_pairs_u64, sort_pairs_u64_static, sort_static_max_n, tangent_balls, version, workspace_bytes,
                  estimate_dtn_both, workspace_bytes_both, estimate_dtn_coo_both, estimate_dtn_host_coo, accumulate_coo, orient_samples_fast, estimate_dtn_batch)

__all__ = ["steklov_eigs", "project_galerkin", "project_galerkin_coo", "winding_number", "orient_samples", "CooMatrix", "PointBasis", "estimate_dtn_coo", "knn_weights", "Bvh", "BvhInfo", "McsError", "Params", "Samples", "Stats", "accumulate", "build_bvh",
           "closest_point", "closest_point_bruteforce", "estimate_dtn_exterior", "estimate_dtn_host",
           "estimate_dtn_interior", "launch_count", "lib",
           "num_records", "philox4x32_10", "profile_enable", "profile_last", "run_walks", "sort_pairs_u64", "sort_pairs_u64_static", "sort_static_max_n", "tangent_balls", "version",
           "workspace_bytes", "estimate_dtn_both", "workspace_bytes_both", "estimate_dtn_coo_both", "estimate_dtn_host_coo", "accumulate_coo", "orient_samples_fast", "estimate_dtn_batch"]
