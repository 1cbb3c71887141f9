"""B200-native (sm_100a) mixed-precision tile Cholesky for Kernel Ridge Regression.

Thin Python binding over the C ABI of include/krr_mp.h (argument marshalling only; every step of
the path runs in the CUDA kernels of csrc/).  PyTorch supplies device memory and streams.
There is no CPU fallback: importing works anywhere, calling needs the built library and a B200.
"""
from .binding import (FP32, FP16, FP8, FLAG_PREROUND_A, FLAG_A_TILED_LOWER, FLAG_NO_LOOKAHEAD, FLAG_FP8_VIA_FP16, FLAG_NO_CTA_PAIRS, FLAG_FUSED_CHAIN, FLAG_KERNEL_IBS, FLAG_KERNEL_LINEAR, FLAG_NO_TAIL_SPLIT, KrrError, Factor,
                      lib, library_path, precision_map, precision_map_static, potrf_mp, potrs, refine, pcg, associate_host, krr_build, build_rr, krr_predict, fit_host, band_map, precision_map_from_build,
                      factor_bytes, factor_tile_offset, tile_slot, uniform_map, last_launch_count,
                      profile_enable, profile_read, profile_timeline, PROFILE_CATEGORIES, Graph, graph_begin, graph_end, potrs_workspace, peak_probe, shutdown, dist_schedule)

__all__ = ["FP32", "FP16", "FP8", "FLAG_PREROUND_A", "FLAG_A_TILED_LOWER", "FLAG_NO_LOOKAHEAD", "FLAG_FP8_VIA_FP16", "FLAG_NO_CTA_PAIRS", "FLAG_FUSED_CHAIN", "FLAG_KERNEL_IBS", "FLAG_KERNEL_LINEAR", "FLAG_NO_TAIL_SPLIT", "KrrError", "Factor",
           "lib", "library_path", "precision_map", "precision_map_static", "potrf_mp", "potrs", "refine", "pcg", "associate_host", "krr_build", "build_rr", "krr_predict", "fit_host", "band_map", "precision_map_from_build",
           "factor_bytes", "factor_tile_offset", "tile_slot", "uniform_map", "last_launch_count",
           "profile_enable", "profile_read", "profile_timeline", "PROFILE_CATEGORIES", "Graph", "graph_begin", "graph_end", "potrs_workspace", "peak_probe", "shutdown", "dist_schedule"]
