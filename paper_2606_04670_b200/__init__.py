"""paper_2606_04670_b200 -- B200-native (sm_100a) hot path of LipFit (arxiv/paper_2606_04670).

The product is the C-ABI library `liblipfit.so` (include/lipfit.h, sources in csrc/); this package
is its thin ctypes binding with the same entry-point names.
"""
from .binding import (LIPFIT_L1, LIPFIT_L2, LIPFIT_LINF, LIPFIT_MAX_DIM, LIPFIT_MAX_K,  # noqa: F401
                      LipfitError, bounds_variant, get_timing, knn_fallbacks, knn_key_error_ratio, knn_set_tensor_cores, knn_variant, launch_count, set_timing, lipfit_bounds,
                      lipfit_bounds_host, lipfit_bounds_pruned, lipfit_smooth_objective_pruned, lipfit_bounds_topk, LIPFIT_MAX_TOPK, lipfit_knn, lipfit_knn_host, lipfit_lbfgs,
                      lipfit_lipschitz_constant, lipfit_lipschitz_constant_host,
                      lipfit_distance_quantiles, lipfit_local_lipschitz, lipfit_values_local, LIPFIT_LOCAL_KNOTS,
                      lipfit_smooth, lipfit_smooth_host, lipfit_smooth_objective, load,
                      status_string, version)
