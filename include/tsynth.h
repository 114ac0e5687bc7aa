/*
 * tsynth.h -- C-ABI boundary of libtsynth.so: batched rendering of the default modular-synth Voice
 * of arXiv 2104.12922 on one B200 (sm_100a).
 *
 * Citations: P:Lnnn = PAPER.md line nnn; S0..S14 / D1..D21 = the step definitions and readings listed
 * in DESIGN.md ("Definition of the path", "Readings"), which restate SURVEY.md section 8(c).
 *
 * Conventions
 *   - Every pointer is a DEVICE pointer unless its name starts with `host_` or the comment says host.
 *   - The caller owns every buffer it passes in.  The library owns only an internal workspace
 *     (control tables; grown on demand, released by ts_shutdown()).
 *   - Calls enqueue work on the stream given to ts_set_stream() (default: the legacy stream 0) and
 *     return without synchronising, except ts_render_host(), ts_sync() and ts_shutdown().
 *   - Return value 0 = TS_OK, negative = error; ts_last_error() gives the text.  No exceptions,
 *     no abort(), nothing printed.
 *   - Hardware behaviour the control stage relies on (reading D28): aligned 16-byte volatile vector accesses
 *     are single transactions on sm_100 (checked on every read by a doubled epoch field: a torn read is retried, never
 *     used), and CTAs are dispatched in linear block-index order (not checkable; a violation surfaces as TS_ECUDA
 *     "look-back timeout" from ts_sync() after a bounded wait, not as wrong audio).
 *   - Not thread-safe: one host thread drives one library instance (one GPU per process).  The library state (nebula,
 *     workspaces, internal streams) is one process-wide singleton: one nebula at a time, one device per process, which
 *     is what one-process-per-GPU launches (torchrun) need.
 */
#ifndef TSYNTH_H
#define TSYNTH_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TS_NPARAM 78 /* parameters of the default Voice */
#define TS_R 100     /* audio rate / control rate, P:L117 (44.1 kHz / 441 Hz); reading D2 */

enum {
    TS_OK = 0,
    TS_EINVAL = -1, /* B <= 0, sr <= 0, seconds <= 0, size overflow, nebula out of supported range */
    TS_ENULL = -2,  /* a required pointer is NULL */
    TS_ECUDA = -3,  /* a CUDA call failed; text in ts_last_error() */
    TS_ENOMEM = -4  /* workspace allocation failed */
};

/* One voice's parameter record (320 B, 16-B aligned).  u[p] in [0,1] is the normalised parameter p
 * ("sampled uniformly from the normalized range"), layout S2; noise_key seeds the voice's
 * white-noise stream ("even of noise oscillators"; reading D4). */
typedef struct {
    float u[TS_NPARAM];
    uint32_t noise_key[2];
} ts_voice;

/* One nebula entry: human range [lo, hi], curve exponent c (u^(1/c), reading D7),
 * symmetric != 0 -> the curve acts on |2u-1| about the centre. */
typedef struct {
    double lo, hi, curve;
    int64_t symmetric;
} ts_range;

typedef struct {
    float *audio;        /* [B][N] row-major fp32, N = ts_num_samples(sr, seconds); required          */
    float *params_human; /* [B][78] mapped parameter values (fp64 result rounded to fp32); may be NULL */
} ts_out;

/* S1 (readings D3, D5).  Voice b of the call is global voice g = batch_index*B + b.
 * key = (seed lo32, seed hi32); Philox4x32-10 block i = 0..19 with counter (i, g lo32, g hi32, 0)
 * gives words 4i..4i+3; u[p] = (word_p >> 8) * 2^-24; noise_key = first two words of the block with
 * counter (0, g lo32, g hi32, 2).  Writes d_params[0..B).  Integer-exact; independent of B (D3). */
int ts_sample_params(uint64_t seed, uint64_t batch_index, int B, ts_voice *d_params);

/* S2..S14 (BASELINE.json north_star).  Renders B voices of `seconds` at `sr` Hz:
 * parameter map -> 6 ADSR + 2 LFO at control ticks (every TS_R samples) -> modulation mixer ->
 * linear upsampling -> phase-accumulating sine and square/saw VCOs + Philox white noise -> VCAs ->
 * mixer -> out.audio.  u outside [0,1] (or NaN) is clamped to [0,1].  d_params is read only.
 * Errors: TS_ENULL (d_params or out.audio NULL), TS_EINVAL (sizes; or the active nebula allows an
 * oscillator increment beyond the supported 2^18/TS_R cycles per sample at this sr: the check is on the nebula's
 * maximum pitch, midi.hi + tune.hi + |depth|, not on the voices of the call, so the default nebula -- 291 cycles per
 * sample at 44.1 kHz -- is refused below sr = 4.9 kHz). */
int ts_render(const ts_voice *d_params, int B, int sr, double seconds, ts_out out);

/* Output sample formats.  The path computes in fp32 (fp64 / Q0.64 for the phase chain) whatever the format; TS_F16 and
 * TS_BF16 round the finished fp32 sample once (round to nearest even) when it is stored, which halves the path's only
 * HBM traffic and the device->host bytes of an end-to-end call ("faster to render ... than to
 * download").  |sample| <= 1.125 (S11), so fp16 never overflows. */
enum { TS_F32 = 0, TS_F16 = 1, TS_BF16 = 2 };

/* ts_render with the output format chosen per call: d_audio is [B][N] of float, __half or __nv_bfloat16 (device). */
int ts_render_fmt(const ts_voice *d_params, int B, int sr, double seconds, int fmt, void *d_audio,
                  float *d_params_human);

/* Convenience end-to-end call with HOST buffers: ts_sample_params + ts_render on the device, then
 * device->host copies of audio ([B][N] fp32) and, if host_params is not NULL, of the ts_voice
 * records.  Synchronises.  Device staging memory belongs to the library workspace. */
int ts_render_host(uint64_t seed, uint64_t batch_index, int B, int sr, double seconds,
                   float *host_audio, ts_voice *host_params);
/* The same with the output format chosen per call (host_audio: [B][N] of float / half / bfloat16). */
int ts_render_host_fmt(uint64_t seed, uint64_t batch_index, int B, int sr, double seconds, int fmt,
                       void *host_audio, ts_voice *host_params);

/* Streaming corpus generation ("generated on the fly from a batch index"; BASELINE.json configs[2]):
 * batches first_batch .. first_batch + n_batches - 1 of B voices each, batch i sampled and rendered into ring slot
 * i % n_ring: records at d_params_ring[(i % n_ring) * B], audio at d_audio_ring[(i % n_ring) * B * N].  Same
 * results as n_batches calls of ts_sample_params + ts_render, but consecutive batches rotate over
 * ts_streaming_lanes() internal lanes (a workspace, a high-priority setup / control stream and a low-priority audio
 * stream each), so the control stage of one batch overlaps the audio stages of the previous ones.  n_ring a multiple
 * of ts_streaming_lanes() keeps every ring slot on one audio stream (no cross-stream events are needed then).  The
 * work is ordered after everything queued on the set stream and the set stream continues after it; the call
 * itself does not synchronise.  A slot is overwritten n_ring batches later: consume it before that. */
int ts_corpus_render(uint64_t seed, uint64_t first_batch, int n_batches, int B, int sr, double seconds,
                     ts_voice *d_params_ring, float *d_audio_ring, int n_ring);

/* ts_corpus_render with the output format chosen per call (d_audio_ring: [n_ring][B][N] of float / half / bfloat16). */
int ts_corpus_render_fmt(uint64_t seed, uint64_t first_batch, int n_batches, int B, int sr, double seconds, int fmt,
                         ts_voice *d_params_ring, void *d_audio_ring, int n_ring);

/* Streaming with ONE NEBULA PER BATCH ("per-call tables per batch"; P:L145 a nebula is the table of
 * (min, max, curve, symmetric) of all parameters; P:L270 the paper's tuning runs render 256 sounds under each of 1000
 * candidate tables, curves log-uniform in [0.1, 10]).  As ts_corpus_render_fmt, but batch i is mapped with
 * host_tables[i * TS_NPARAM .. (i + 1) * TS_NPARAM): same results as ts_set_nebula(table i) + ts_sample_params +
 * ts_render per batch, with the batches overlapping on the streaming lanes.  All tables are checked first (TS_EINVAL as
 * ts_set_nebula and ts_render would return, nothing launched) and uploaded once; host_tables may be freed when the call
 * returns.  The active nebula (ts_set_nebula) is not changed by the call. */
int ts_corpus_render_nebulae(uint64_t seed, uint64_t first_batch, int n_batches, int B, int sr, double seconds, int fmt,
                             const ts_range *host_tables, ts_voice *d_params_ring, void *d_audio_ring, int n_ring);

/* Streaming corpus ITERATOR ("generated on the fly", P:L98 sounds paired with their
 * parameters, P:L102 train/test blocks).  ts_corpus_open() fixes the corpus (seed, B, sr, seconds, format), the caller's
 * ring of n_ring >= 2 output slots and the first batch index, and starts rendering n_ring - 1 batches ahead on the
 * library's internal streams.  Each ts_corpus_next() hands out the next batch: the slot's device pointers, the batch
 * index, the global index of its first voice (g = batch_index * B) and the train/test designation of its first and last
 * voice (equal whenever B divides 1024; a batch of 1024-aligned voices never straddles a block).  The call makes the set stream wait
 * for that batch (no host synchronisation) and re-arms the slot handed out by the PREVIOUS call with the batch
 * n_ring - 1 ahead, ordered after everything the caller has queued on the set stream so far: consume a batch on the set
 * stream before asking for the next one.  ts_corpus_close() drains the internal streams.
 * While an iterator is open the nebula is fixed: ts_set_nebula, ts_corpus_render*, ts_render_r return TS_EINVAL.  If a
 * batch cannot be issued (TS_ENOMEM, TS_ECUDA), ts_corpus_open / ts_corpus_next drain the internal streams and CLOSE the
 * iterator before returning that error: there is never a half-open iterator to clean up. */
typedef struct {
    uint64_t seed;
    int B, sr;
    double seconds;
    int fmt;                 /* TS_F32 / TS_F16 / TS_BF16 */
    int n_ring;              /* >= 2 */
    void *d_audio_ring;      /* [n_ring][B][N] in fmt (device, caller-owned) */
    ts_voice *d_params_ring; /* [n_ring][B] records (device, caller-owned) */
} ts_corpus_cfg;
typedef struct {
    void *d_audio;           /* [B][N] in the corpus format */
    ts_voice *d_params;      /* [B] records: normalised parameters + noise keys */
    uint64_t batch_index;
    uint64_t first_voice;    /* global voice index of row 0 */
    int is_test_first, is_test_last; /* ts_corpus_is_test of the first and the last voice of the batch */
    int slot;
} ts_corpus_batch;
int ts_corpus_open(const ts_corpus_cfg *host_cfg, uint64_t first_batch);
int ts_corpus_next(ts_corpus_batch *host_out);
int ts_corpus_close(void);

/* Control-rate rendering on its own (P:L117 control modules at 1/100 of the audio rate; the paper's Fig. 2 workload,
 * P:L131): the five modulation-mixer rows (S5..S7: six ADSRs, two LFOs, mixer) at the K = ts_num_ticks(N) control
 * ticks -> d_ctl[B][5][K] fp64, rows M_0 (vco1 pitch), M_1 (vco1 amp), M_2 (vco2 pitch), M_3 (vco2 amp),
 * M_4 (noise amp).  Ticks after the voice has gone silent for good are written as 0.  No audio is rendered and nothing
 * of the oscillator stage runs (no interval sums, no phase scan, no control table). */
int ts_render_controls(const ts_voice *d_params, int B, int sr, double seconds, double *d_ctl);
/* The same with the tick spacing chosen per call: one tick every R >= 1 samples (control rate sr / R, reading D2 with R
 * in place of 100); K = ts_num_ticks_r(N, R) = ceil(N / R) + 1.  R = 1 is the audio-rate-control mode of SURVEY 8(f)
 * item 3 (upsampling is then the identity, pin P7): every ADSR / LFO / mixer value is evaluated at every sample. */
int ts_render_controls_r(const ts_voice *d_params, int B, int sr, double seconds, int R, double *d_ctl);
int64_t ts_num_ticks_r(int64_t N, int R);

/* ts_render with the tick spacing chosen per call, fp32 output: R = TS_R is ts_render; R = 1 is the audio-rate-control
 * mode of SURVEY 8(f) item 3 (every sample is a control tick: ADSRs, LFOs and the mixer are evaluated at every sample,
 * upsampling is the identity, pin P7; reading D27).  R = 1 is a mode for studying the two-rate design (D1), not the hot
 * path: its control table has one entry per sample (80 B), so a call is split into chunks of a few voices.  Other values
 * of R: TS_EINVAL. */
int ts_render_r(const ts_voice *d_params, int B, int sr, double seconds, int R, float *d_audio);

/* Maximum mean discrepancy of two sets of n embeddings of dimension d with the l1 distance as the core distance
 * (Eq. 2 at P:L230; "1/nn" there is read as 1/n^2, reading D25; the paper's setting is n = 1000, d = 512,
 * P:L257):  MMD(X, Y) = (1/n^2) sum_{i,j} [ 2 |x_i - y_j|_1 - |x_i - x_j|_1 - |y_i - y_j|_1 ].
 * d_x, d_y: [n][d] fp32 row-major (device), finite values.  d_out (device, 4 doubles): [0] MMD, [1] sum_ij |x_i - y_j|_1,
 * [2] sum_ij |x_i - x_j|_1, [3] sum_ij |y_i - y_j|_1.
 * Two forms, the same result up to their rounding:
 * ts_mmd_l1_pairwise, O(d n^2): fp32 differences and per-pair sums over 64 x 64 tiles of pairs, fp64 sums over pairs in a
 *   fixed order.
 * ts_mmd_l1_sorted, O(d n log^2 n), n <= 8192 (beyond that it runs the pairwise form): it never forms a pair -- the three
 *   sums decompose over the d components, and the sum of |a - b| over all pairs of ONE component follows from one sort of
 *   its 2n values (every value against the count and the sum of the smaller ones).  The values of a component are taken
 *   on a fixed-point grid of 2^-61 of its largest magnitude (an fp32 value is on the grid unless it is 2^37 times smaller
 *   than that maximum) and everything after that is exact integer arithmetic.
 * ts_mmd_l1 runs whichever is faster at this n (the paper's n = 1000, d = 512: sorted, 80 vs 110 us on a B200; n = 4000:
 *   336 vs 1466 us; n = 256: pairwise).  All three are bitwise reproducible (fixed summation orders).  MMD(X, X) == 0
 *   EXACTLY is a property of the sorted form (integer sums: the three pair sums of X = Y are the same integer).  The
 *   pairwise form adds the cross matrix and the two symmetric ones in different orders (all tiles vs doubled upper
 *   triangle), so its MMD(X, X) is 0 only while the fp64 sums of the fp32 pair sums are still exact (roughly
 *   24 + log2(n^2) + the dynamic range of the pair sums <= 53 bits); beyond that it is 0 to within fp64 rounding of sums
 *   of that size.  ts_mmd_l1 runs the pairwise form for n > 8192 and for small n.
 * Errors: TS_ENULL, TS_EINVAL (n <= 0, d <= 0, n > 65535). */
int ts_mmd_l1(const float *d_x, const float *d_y, int n, int d, double *d_out);
int ts_mmd_l1_pairwise(const float *d_x, const float *d_y, int n, int d, double *d_out);
int ts_mmd_l1_sorted(const float *d_x, const float *d_y, int n, int d, double *d_out);

/* ts_mmd_l1 for callers that cannot allocate device memory at call time.  The three calls above keep their per-CTA
 * partial sums in a workspace obtained with cudaMalloc (grown on demand, freed by ts_shutdown()).  That does not suit
 * every host of this library:
 *   - a process in which another allocator already owns the whole GPU (for example a framework's caching pool that was
 *     sized to all of HBM), so that a raw cudaMalloc has nothing left to return;
 *   - a real-time audio or serving loop, where cudaMalloc / cudaFree may synchronise the whole device and take an
 *     unbounded time in the middle of a deadline;
 *   - an embedding host (plug-in, sandboxed worker) whose rules forbid allocating after start-up.
 * ts_mmd_l1_static runs the same kernels as ts_mmd_l1 (the faster form at this n) and returns the same bits, but its
 * scratch is a fixed array that is part of the library's device image: TS_MMD_STATIC_MAX_PARTIALS doubles = 256 KB,
 * resident on every GPU that loads libtsynth.so from load to process exit, used or not.  The call itself makes no
 * cudaMalloc, cudaFree or other allocating call; d_x, d_y and d_out are the caller's, as above.
 * Limit: max(3 d, 4 (2 T^2 + T)) <= TS_MMD_STATIC_MAX_PARTIALS with T = ceil(n / 64), i.e. n <= 4032 and d <= 10922 (the
 *   paper's n = 1000, d = 512 needs 2112).  Anything larger: TS_EINVAL with the sizes in ts_last_error(), nothing launched.
 * First call on a device: it looks up the array's device address (once per device, which must be the current device;
 *   that is the only set-up).  Make that first call during start-up, before any stream capture begins; later calls only
 *   launch the two kernels on the ts_set_stream() stream.
 * Sharing: every call on a device uses the same array and leaves its partial sums there.  Nothing needs clearing between
 *   calls (each call overwrites every entry it later reads), but two calls that can run on the GPU at the same time --
 *   different streams, or different host threads -- race on it and give garbage.  Calls issued on one stream are ordered
 *   and safe.  It does not share anything with ts_mmd_l1's workspace, so those calls may overlap with this one.
 * Errors: TS_ENULL, TS_EINVAL (n <= 0, d <= 0, n > 65535, beyond the limit), TS_ECUDA. */
#define TS_MMD_STATIC_MAX_PARTIALS 32768
int ts_mmd_l1_static(const float *d_x, const float *d_y, int n, int d, double *d_out);

/* Train/test designation of global voice g ("9 * 1024 samples are designated as train, the next 1024
 * samples as test, etc.", i.e. one tenth of the corpus): 1 if (g / 1024) % 10 == 9, else 0.  A position in
 * the corpus, so it is the same for batch size 128 and 1024 (D3).  Host function, no GPU work. */
int ts_corpus_is_test(uint64_t g);

/* D17: N = llround(sr*seconds);  S5: K = ceil(N/TS_R) + 1 control ticks. */
int64_t ts_num_samples(int sr, double seconds);
int64_t ts_num_ticks(int64_t N);
int ts_streaming_lanes(void);                     /* lanes the streaming calls rotate batches over (3) */

int ts_set_stream(void *cuda_stream);              /* cudaStream_t; NULL = legacy default stream   */
int ts_default_nebula(ts_range host_out78[TS_NPARAM]); /* host copy of the built-in table S2        */
int ts_set_nebula(const ts_range *host_in78);      /* host table; NULL restores the default.  TS_EINVAL: non-finite entries, curve <= 0, a negative range for a weight (LFO shapes 35..39, 43..47; modulation mixer 48..67), or a corpus iterator is open (its nebula is the one active at ts_corpus_open; close it first) */
size_t ts_workspace_bytes(int B, int sr, double seconds); /* device bytes ts_render will hold      */
const char *ts_last_error(void);                   /* host string, owned by the library            */
int ts_sync(void);                                 /* cudaStreamSynchronize on the set stream; TS_ECUDA if a kernel raised the device error flag */
void ts_shutdown(void);                            /* frees the workspace                          */

/* Per-kernel device times of the LAST ts_render when timing is enabled (CUDA events on the set
 * stream around each kernel; costs a few microseconds per call, so off by default).
 * host_ms[0] = control kernel, host_ms[1] = audio kernel, summed over voice chunks; synchronises. */
int ts_set_timing(int enable);
int ts_last_kernel_ms(float host_ms[2]);
/* The measurement aids bench.py's roofline numbers come from (ts_time_*) are NOT part of this library: they are declared in
 * tsynth_measure.h and exist only in libtsynth_measure.so, the same sources built with -DTS_MEASURE. */
/* Counters of the LAST ts_render (host): [0] kernels launched, [1] voice chunks,
 * [2] audio samples in the active (non-silent) prefix summed over voices (counted only while timing is
 * enabled with ts_set_timing; valid after ts_sync). */
int ts_last_stats(int64_t host_stats[3]);

/* Debug exports used only by the parity tests. */
/* S12: words n0..n0+count-1 of the noise stream of `key` (host array of 2) -> d_out[count]. */
int ts_debug_noise_u32(const uint32_t host_key[2], uint64_t n0, int count, uint32_t *d_out);
/* The five modulation-mixer rows as the AUDIO path computes them (same launch as ts_render up to the control table,
 * every tick evaluated) -> d_ctl[B][5][K] fp64. */
int ts_debug_controls(const ts_voice *d_params, int B, int sr, double seconds, double *d_ctl);
/* S9: phase of VCO `vco` (1 or 2) at every sample, cycles in [0,1) -> d_phase[B][N] fp64. */
int ts_debug_phase(const ts_voice *d_params, int B, int sr, double seconds, int vco, double *d_phase);

#ifdef __cplusplus
}
#endif
#endif /* TSYNTH_H */
