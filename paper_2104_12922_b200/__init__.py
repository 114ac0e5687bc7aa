"""paper_2104_12922_b200 -- batched rendering of the arXiv 2104.12922 modular-synth Voice on B200.

The product is the C-ABI library libtsynth.so (include/tsynth.h, sources under csrc/).  This package is
its thin Python binding: argument marshalling only, every step of the path runs in the CUDA kernels.
There is no CPU fallback: importing `binding` fails loudly if the library has not been built.
"""
from .binding import (NPARAM, R, NEBULA_DTYPE, TS_F32, TS_F16, TS_BF16, TsynthError, lib, lib_path, use_measure_build, ts_sample_params,  # noqa: F401
                      ts_render, ts_render_fmt, ts_render_host, ts_render_host_fmt, ts_corpus_render, ts_corpus_render_fmt, ts_corpus_render_nebulae,
                      ts_corpus_open, ts_corpus_next, ts_corpus_close, ts_corpus_is_test, ts_num_samples, ts_num_ticks,
                      ts_num_ticks_r, ts_streaming_lanes, ts_set_stream, ts_default_nebula, ts_set_nebula, ts_workspace_bytes, ts_sync, ts_shutdown,
                      ts_set_timing, ts_time_kernels, ts_time_audio_lanes, ts_time_fill, ts_time_alu_bound, ts_time_pipes, ts_last_kernel_ms, ts_last_stats, ts_render_r, ts_render_controls,
                      ts_render_controls_r, ts_mmd_l1, ts_mmd_l1_static, MMD_STATIC_MAX_PARTIALS, ts_debug_noise_u32, ts_debug_controls, ts_debug_phase)
