// ts_common.cuh -- shared device-side definitions of libtsynth (CUDA path only; the CPU oracle
// under oracle/ shares nothing with this file).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tsynth.h"

// ---- geometry of the audio kernel --------------------------------------------------------------
// One thread renders one RUN of consecutive samples; five runs make one control interval (TS_R).
constexpr int TS_RUN = 20;                    // samples per thread (5 float4 groups, 5 Philox blocks)
constexpr int TS_RUNS_PER_TICK = TS_R / TS_RUN;
constexpr int TS_AUDIO_THREADS = 128;         // threads per CTA of the audio kernel
constexpr int TS_TILE = TS_AUDIO_THREADS * TS_RUN;  // 2560 samples = 10 240 B staged in smem per CTA

// ---- control table: one entry per control tick, written by the control kernel ------------------
// phi  : VCO phase at the tick's first sample, cycles in [0,1)            (S9, exact integer scan)
// inc  : phase increment of that sample, cycles/sample                    (S9)
// e1   : rho - 1, rho = per-sample ratio of increments inside the interval (pitch is linear in n)
// g20  : sum_{i<20} rho^i  (so that a run starting 20 samples later has phi += w*g20, w *= 1+e1*g20)
// a1..a3 : VCA gains at the tick with the mixer level / level sum (and 1 - s/2 for VCO2) folded in
struct __align__(16) ts_tick {
    double phi1, inc1, e1_1, g20_1;
    double phi2, inc2, e1_2, g20_2;
    float a1, a2, a3, pad;
};
static_assert(sizeof(ts_tick) == 80, "ts_tick layout");

// ---- per-voice header written by the control kernel -------------------------------------------
struct __align__(16) ts_vhdr {
    float shape;      // s of S11
    float tanh_c;     // (pi/2) * k * 2*log2(e): tanh(x) = 1 - 2/(1 + 2^(tanh_c * sin(theta)))
    uint32_t nk0, nk1;
    int32_t n_act;    // samples [n_act, N) are exactly 0 (multiple of TS_R, or N)
    int32_t n_ticks;  // table entries [0, n_ticks) are valid
    int32_t pad[2];   // pad[0] != 0: steepness k <= 512, the audio kernel takes the square/saw from MUFU.SIN / MUFU.COS on the whole cycle
};
static_assert(sizeof(ts_vhdr) == 32, "ts_vhdr layout");

// ---- per-voice constants: written once per voice by the setup kernel, staged in shared memory by every live
// chunk CTA of the control kernel -------------------------------------------------------------------------
struct __align__(16) ts_voice_consts {
    double h[TS_NPARAM + 2];  // mapped parameters (S2 layout)
    double rs[18], rd[18], rinv[18];  // per ADSR the three ramps (release, attack, decay): start, duration, 1/duration
    double lfo_w[2][5];       // LFO shape weights / their sum (0 if the sum is 0)
    double mix_w[5][4];       // modulation-mixer weights / their row sum
    double dq_f[2], dq_d[2];  // LFO frequency / cr and rate-mod depth / cr (cycles per tick)
    double g[3];              // VCA gains: mixer level / level sum; VCO2 also carries (1 - s/2) of S11
    int jsil;                 // first tick at which the voice is silent for good (== K if never)
    int slow;                 // some ADSR alpha <= 0: use the generic power
    int pad[2];
};
static_assert(sizeof(ts_voice_consts) % 16 == 0, "ts_voice_consts is copied in 16-byte pieces");

// ---- S0 Philox4x32-10 ---------------------------------------------------------------------------
__device__ __forceinline__ void ts_philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                 uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        if (r > 0) {
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// launchers (host), one per .cu file
cudaError_t ts_launch_sample(uint64_t seed, uint64_t g0, int B, ts_voice *d_params, cudaStream_t st);
cudaError_t ts_launch_noise_debug(uint32_t k0, uint32_t k1, uint64_t n0, int count, uint32_t *d_out, cudaStream_t st);
cudaError_t ts_upload_nebula(const ts_range *host78, cudaStream_t st);
cudaError_t ts_upload_math_tables(cudaStream_t st);
size_t ts_control_agg_bytes(int B, int K);  // look-back slots; must be zero before the first launch
// the audio-rate-control mode: table entries are per SAMPLE (control kernel with R = 1)
cudaError_t ts_launch_audio_r1(const ts_tick *table, const ts_vhdr *hdr, int B, int64_t N, int K, float *audio, cudaStream_t st);
cudaError_t ts_launch_body_bench(int fastsin, int reps, float *d_sink, cudaStream_t st);  // the audio kernel's sample loop alone
cudaError_t ts_launch_fill(void *d_dst, size_t bytes, cudaStream_t st);  // store-only fill kernel (measurement aid)
constexpr int TS_NPIPES = 8;
cudaError_t ts_measure_pipes(double host_rates[TS_NPIPES], cudaStream_t st);  // issue rates of the audio kernel's instruction kinds
// pairwise: 0 = whichever form is faster at this n, 1 = the O(d n^2) tiled form, 2 = the sorted form (n <= 8192, else tiled)
cudaError_t ts_launch_mmd(const float *d_x, const float *d_y, int n, int d, double *d_partial, double *d_out, int pairwise, cudaStream_t st);
size_t ts_mmd_partial_count(int n, int d);
// ts_mmd_l1_static: the faster form with the partial sums in the module's own static device array (no allocation)
size_t ts_mmd_static_capacity();  // partial sums the array holds (TS_MMD_STATIC_MAX_PARTIALS)
cudaError_t ts_launch_mmd_static(const float *d_x, const float *d_y, int n, int d, double *d_out, cudaStream_t st);
// epoch: a value never used before on this `agg` buffer (flags from older launches then read as "not ready")
// Per-voice setup (S1 optional, S2/S3, derived constants, last audible tick, header).  sample != 0: draw the records
// first (S1, global voices g0 .. g0 + B - 1 under `seed`) and write them to d_params; else read d_params.
// R: samples per control tick (TS_R on the audio path; any R >= 1 for control-rate rendering on its own)
cudaError_t ts_launch_setup(ts_voice *d_params, int sample, uint64_t seed, uint64_t g0, int B, int sr, int R, int64_t N, int K,
                            ts_voice_consts *vc, ts_vhdr *hdr, float *params_human, unsigned long long *d_active, int full,
                            const void *d_nebula, cudaStream_t st);  // d_nebula: a table in the device layout, NULL = the active nebula
size_t ts_nebula_device_bytes();                                           // bytes of one table in the device layout
void ts_nebula_to_device_layout(const ts_range *host78, void *out);       // host-side conversion (adds 1 / curve)
// phases != 0: also the S9 tick-level phase scan and the control table (needed by the audio kernel); phases == 0 stops
// after the modulation mixer (control-rate rendering on its own).  n_audible_max >= 0: no voice is audible at or after this sample (chunks past it are not launched); d_err: device flag raised if a look-back wait gives up
cudaError_t ts_launch_control(const ts_voice_consts *vc, int B, int sr, int R, int64_t N, int K, ts_tick *table, void *agg,
                              unsigned int epoch, double *dbg_ctl, int phases, int64_t n_audible_max, unsigned int *d_err, cudaStream_t st);
// mode 0: audio; mode 1 / 2: write the phase of VCO 1 / 2 (fp64 cycles) to dbg_phase instead.
// tails != 0: long silent tails are expected (nebula + buffer length), let the audible CTAs write them asynchronously;
// n_audible_max: no voice is audible at or after this sample (then no CTA is launched for those tiles)
// fmt: TS_F32 / TS_F16 / TS_BF16 output samples
cudaError_t ts_launch_audio(const ts_tick *table, const ts_vhdr *hdr, int B, int64_t N, int K, void *audio, int fmt,
                            int mode, int tails, int64_t n_audible_max, double *dbg_phase, cudaStream_t st);
