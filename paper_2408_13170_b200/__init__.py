"""B200-native semi-coherent statistic (hot path of arXiv 2408.13170): thin Python binding over libscstat.so.

Every step of the path runs in the CUDA kernels of csrc/; this package only marshals arguments.
There is no CPU fallback: importing works anywhere, but every call needs the built library and a CUDA device.
"""
from .binding import (SCError, ScConfig, ScSearchConfig, Handle, sc_pso_step_labeled, sc_kmeans, sc_kmeans_static, SC_KMEANS_STATIC_MAX_K, sc_search_run, sc_whiten_streams, sc_eval_stat_streams, load_library, library_path, sc_init_data, sc_init_data_host, sc_init_data3, sc_gen_template3,
                      sc_eval_stat, sc_eval_stat_host, sc_eval_segments, sc_eval_stat_adaptive, sc_eval_components, sc_eval_loglike, sc_data_norm,
                      sc_gen_template, sc_pso_step, sc_pso_best, sc_pso_pick, sc_pso_move,
                      sc_get_counters, sc_get_launch_info, sc_get_timing, sc_measure_fp64_peak, sc_set_option, sc_free, sc_last_error, sc_version,
                      SC_OPT_PRECISION, SC_OPT_F32_MIN_SEG, SC_OPT_SCRATCH_BYTES, SC_OPT_TC_MAX_S,
                      SC_OPT_STRIDE_LOG2, SC_OPT_PROFILE, SC_OPT_SINCOS, SC_OPT_MUFU_MIN_SEG, SC_OPT_ESCALATE,
                      SC_OPT_ESC_TAU_POLY_X1000, SC_OPT_ESC_TAU_MUFU_X1000, SC_OPT_WINDOW_SORT, SC_OPT_TENSOR_CORES, SC_OPT_FUSED_AET, SC_OPT_WINDOW_FRACTION_PPM, SC_OPT_QUAD_AMPLITUDES, SC_FLAVOUR_MUFU, SC_FLAVOUR_MERGE, SC_FLAVOUR_QUAD, SC_FLAVOUR_TC, SC_FLAVOUR_AET,
                      EXPORTED_SYMBOLS)

__all__ = ["SCError", "ScConfig", "ScSearchConfig", "Handle", "sc_pso_step_labeled", "sc_kmeans", "sc_kmeans_static", "SC_KMEANS_STATIC_MAX_K", "sc_search_run", "sc_whiten_streams", "sc_eval_stat_streams", "load_library", "library_path", "sc_init_data", "sc_init_data_host", "sc_init_data3", "sc_gen_template3",
           "sc_eval_stat", "sc_eval_stat_host", "sc_eval_segments", "sc_eval_stat_adaptive", "sc_eval_components", "sc_eval_loglike", "sc_data_norm",
           "sc_gen_template", "sc_pso_step", "sc_pso_best", "sc_pso_pick", "sc_pso_move",
           "sc_get_counters", "sc_get_launch_info", "sc_get_timing", "sc_measure_fp64_peak", "sc_set_option", "sc_free", "sc_last_error", "sc_version",
           "SC_OPT_PRECISION", "SC_OPT_F32_MIN_SEG", "SC_OPT_SCRATCH_BYTES", "SC_OPT_TC_MAX_S", "SC_OPT_STRIDE_LOG2", "SC_OPT_PROFILE", "SC_OPT_SINCOS", "SC_OPT_MUFU_MIN_SEG", "SC_OPT_ESCALATE", "SC_OPT_ESC_TAU_POLY_X1000", "SC_OPT_ESC_TAU_MUFU_X1000", "SC_OPT_WINDOW_SORT", "SC_OPT_TENSOR_CORES", "SC_OPT_FUSED_AET", "SC_OPT_WINDOW_FRACTION_PPM", "SC_OPT_QUAD_AMPLITUDES",
           "SC_FLAVOUR_MUFU", "SC_FLAVOUR_MERGE", "SC_FLAVOUR_QUAD", "SC_FLAVOUR_TC", "SC_FLAVOUR_AET", "EXPORTED_SYMBOLS"]
