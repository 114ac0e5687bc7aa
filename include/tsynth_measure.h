/*
 * tsynth_measure.h -- measurement aids for bench.py: what the roofline numbers of the bench line are made from.
 *
 * NOT part of the product ABI (SURVEY 8(b) lists no such call).  These entry points exist only in libtsynth_measure.so:
 * the sources of libtsynth.so plus csrc/ts_measure.cu, compiled with -DTS_MEASURE (paper_2104_12922_b200/build.py builds
 * both).  That library also exports everything tsynth.h declares -- the same kernels, compiled from the same files -- so
 * a process that measures loads it INSTEAD of libtsynth.so (binding.use_measure_build()), and what is timed is the
 * product's own code.  libtsynth.so carries none of this: no ts_time_* symbol, no bench kernel.
 * Conventions as in tsynth.h (device pointers unless named host_, TS_* return codes, ts_last_error()).
 */
#ifndef TSYNTH_MEASURE_H
#define TSYNTH_MEASURE_H

#include "tsynth.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Average device time per launch of the two render kernels on this batch: `reps` back-to-back launches of the
 * control kernel, then `reps` of the audio kernel (output rotating over the n_ring slots of d_audio_ring,
 * [n_ring][B][N] fp32, so that consecutive launches do not rewrite lines still in L2), each group between one pair
 * of CUDA events on the set stream.  host_ms[0] = control, host_ms[1] = audio, milliseconds per launch.
 * A batch that ts_render splits into several voice chunks is timed chunk by chunk and summed.  Synchronises. */
int ts_time_kernels(const ts_voice *d_params, int B, int sr, double seconds, float *d_audio_ring, int n_ring, int reps,
                    float host_ms[2]);
/* Measurement aid: the audio kernel as the streaming calls launch it -- `reps` launches rotating over the
 * ts_streaming_lanes() low-priority audio streams, so that the ramp and drain of one
 * launch (3.8 us for any kernel of this shape) are covered by the other streams' launches -- timed as one interval on the
 * set stream.  *host_ms = interval / reps: an inverse
 * throughput, NOT a launch duration (ts_time_kernels gives that); the difference is the part of a launch in which the SMs
 * hold no CTA.  The batch must fit one voice chunk.  Synchronises. */
int ts_time_audio_lanes(const ts_voice *d_params, int B, int sr, double seconds, float *d_audio_ring, int n_ring,
                              int reps, float *host_ms);
/* Measurement aid: average device time of a store-only kernel (128-bit stores of zeros over d_dst[0 .. bytes)), `reps`
 * launches between one pair of CUDA events on the set stream -> *host_ms per launch.  What a pure store stream reaches on
 * this GPU, quoted beside the copy peak the roofline uses.  Synchronises. */
int ts_time_fill(void *d_dst, size_t bytes, int reps, float *host_ms);
/* Measurement aid: the ALU bound of the audible part, measured.  Runs the audio kernel's own sample loop (S9..S14: the
 * same device function, 20 samples per thread and pass, `reps` passes) with no control table, no global stores and no CTA
 * turnover at 8 warps per SM sub-partition, and returns the audible samples per second the SM pipes sustain with that
 * instruction mix (fastsin: the MUFU.SIN variant of the square/saw sine taken by voices with k <= 512, else the
 * polynomial one).  Synchronises. */
int ts_time_alu_bound(int fastsin, int reps, double *host_samples_per_s);
/* Measurement aid: issue rate of the instruction kinds the audio kernel is made of, each alone, 8 warps per SM
 * sub-partition with 8 independent chains per thread.  host_rates[k] = cycles per warp instruction per sub-partition:
 * [0] FFMA, [1] FFMA2 (packed fp32x2), [2] IMAD.WIDE.U32 (the Philox multiply), [3] LOP3, [4] DFMA, [5] MUFU.SIN with its
 * range-reduction FMUL, [6] MUFU.EX2, [7] I2FP.  DESIGN.md 5.2 derives the kernel's pipe budget from them.  Synchronises. */
int ts_time_pipes(double host_rates[8]);

#ifdef __cplusplus
}
#endif
#endif /* TSYNTH_MEASURE_H */
