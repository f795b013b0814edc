"""B200-native hot path of the 2HOT hashed oct-tree method (arXiv:1310.4502).

Thin binding of the C ABI in ``include/hot.h`` (``libhot.so``, CUDA for sm_100a): argument
marshalling only.  Every step of the path runs in the library's kernels; PyTorch supplies device
buffers and the stream.  There is no CPU fallback: calls raise if the library is missing.

    import torch, paper_1310_4502_b200 as hot
    hot.hot_build(pos, mass, box_lo, box_size, periodic=False)   # pos [n,3], mass [n] cuda fp32
    acc, pot = hot.hot_forces(theta=0.5, eps=1e-3, order=2)
    print(hot.hot_stats())
"""
from __future__ import annotations

from .binding import (HotError, hot_build, hot_export_cells, hot_export_groups, hot_export_keys, hot_export_lists, hot_export_group_orders, hot_forces_tol,
                      hot_export_moments, hot_forces, hot_free, hot_last_error, hot_lookup_keys,
                      hot_far_coefficients, hot_measure_fp32, hot_measure_fp32_operands, hot_set_list_arena, hot_set_softening, hot_sort_keys_noalloc, hot_noalloc_last_error, hot_set_background, hot_kick_drift, hot_set_params, hot_set_stream, hot_stats, hot_step_host, library_path)

__all__ = ["HotError", "hot_build", "hot_forces", "hot_stats", "hot_step_host", "hot_set_params", "hot_set_list_arena", "hot_set_softening", "hot_sort_keys_noalloc", "hot_noalloc_last_error", "hot_set_background", "hot_kick_drift", "hot_far_coefficients", "hot_measure_fp32", "hot_measure_fp32_operands",
           "hot_set_stream", "hot_free", "hot_last_error", "hot_export_keys", "hot_export_cells",
           "hot_export_groups", "hot_export_lists", "hot_export_group_orders", "hot_forces_tol", "hot_export_moments", "hot_lookup_keys", "library_path"]
