// ts_api.cu -- the C-ABI of include/tsynth.h: argument checks, the nebula, the workspace (control tables
// sized to stay L2-resident), voice chunking, kernel launches and the streaming iterator.  No arithmetic of the
// method lives here.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include "ts_common.cuh"
#ifdef TS_MEASURE
#include "../../include/tsynth_measure.h"
#endif

namespace {

// A lane = a workspace with the stream(s) that use it, so that several batches can be in flight at once.
// Lane 0 serves ts_render / ts_render_host on the caller's stream.  Lanes 1 .. TS_SL serve the streaming calls: each
// has a HIGH-priority stream for the (latency-bound) setup and control kernels and a LOW-priority stream for the
// (issue-bound) audio kernel, so that the control stage of batch i+1 is dispatched into the SMs while the audio
// stages of batches i, i-1 still run and fills the issue slots they leave idle.
struct ts_lane {
    cudaStream_t stream = nullptr;
    void *ws = nullptr;
    size_t ws_bytes = 0;
    int lay_B = 0, lay_K = 0;  // layout the look-back slots were last cleared for
    size_t lay_off = 0;
    unsigned int epoch = 0;    // look-back flag value of the latest control launch on this workspace
    unsigned long long *d_active = nullptr;
    unsigned long long *h_active = nullptr;  // pinned
    unsigned int *d_err = nullptr;           // raised by a kernel whose look-back wait gave up
    unsigned int *h_err = nullptr;           // pinned
    // streaming lanes: the audio kernel goes to its own low-priority stream
    cudaStream_t audio_stream = nullptr;
    cudaEvent_t ctl_done = nullptr, aud_done = nullptr;
    bool aud_pending = false;  // aud_done was recorded after the latest audio kernel that reads this workspace
};
#ifndef TS_SLANES
#define TS_SLANES 3  // measured on C2: 2 lanes 32.3 us per step, 3 lanes 26.9, 4 lanes 27.1
#endif
constexpr int TS_SL = TS_SLANES;     // streaming lanes (each: a workspace, a high- and a low-priority stream)
constexpr int TS_LANES = 1 + TS_SL;
constexpr int TS_MAX_RING = 64;

struct ts_corpus_state {  // the streaming iterator (ts_corpus_open / next / close)
    bool open = false;
    ts_corpus_cfg cfg;
    int64_t N = 0;
    uint64_t first = 0, next_out = 0, next_render = 0;  // batch indices
    cudaEvent_t ready[TS_MAX_RING] = {};     // slot rendered
    cudaEvent_t consumed = nullptr;          // the caller's stream has passed the previous hand-out
};

struct ts_state {
    char err[512] = "";
    ts_range nebula[TS_NPARAM];
    bool nebula_init = false;
    bool nebula_dirty = true;  // device copy is stale
    bool math_uploaded = false;
    ts_lane lane[TS_LANES];
    ts_lane *cur = &lane[0];
    cudaEvent_t fork = nullptr;
    // the streaming calls' internal streams: one high-priority (setup, control) and one low-priority (audio) stream per
    // streaming lane, so that consecutive chunks overlap completely (kernel launch gaps included)
    cudaStream_t hi[TS_SL] = {}, lo[TS_SL] = {};
    cudaEvent_t batch_done[TS_MAX_RING][TS_SL] = {};  // audio of batch (count % TS_MAX_RING) issued on lo[x] has finished
    cudaEvent_t join_ev[2 * TS_SL] = {};
    // host staging for ts_render_host
    void *stage = nullptr;
    size_t stage_bytes = 0;
    double *mmd_ws = nullptr;
    size_t mmd_ws_count = 0;
    // per-batch nebulae of ts_corpus_render_nebulae: all tables of a call in the device layout, uploaded once
    void *d_tables = nullptr, *h_tables = nullptr;  // h_tables: pinned
    size_t tables_bytes = 0;
    cudaEvent_t tables_up = nullptr;                // the upload of the latest call has executed
    const void *batch_table = nullptr;              // the table of the batch being issued (NULL: the active nebula)
    // timing / stats
    bool timing = false;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    float ms[2] = {0.f, 0.f};
    int64_t stats[3] = {0, 0, 0};
    ts_corpus_state corpus;
};
ts_state S;

// Control-table budget per voice chunk: small enough to live in the 126 MB L2 next to the audio being
// written, so the audio kernel's table reads never go to HBM.
constexpr size_t TS_TABLE_BUDGET = 48u << 20;

int fail(int code, const char *fmt, const char *detail = "") {
    snprintf(S.err, sizeof S.err, fmt, detail);
    return code;
}
int cuda_fail(cudaError_t e, const char *where) {
    snprintf(S.err, sizeof S.err, "%s: %s", where, cudaGetErrorString(e));
    return TS_ECUDA;
}
#define TS_CUDA(call)                                      \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)

bool fmt_ok(int fmt) { return fmt == TS_F32 || fmt == TS_F16 || fmt == TS_BF16; }
size_t fmt_bytes(int fmt) { return (fmt == TS_F32) ? 4 : 2; }

void default_nebula(ts_range *n) {  // table S2 (D6, D8); ranges from BASELINE.json configs[0]
    auto set = [&](int i, double lo, double hi, double c, int sym) { n[i] = ts_range{lo, hi, c, sym}; };
    set(0, 0.0, 127.0, 1.0, 0);
    set(1, 0.01, 1.0, 0.5, 0);
    for (int e = 0; e < 6; ++e) {
        const int b = 2 + 5 * e;
        set(b + 0, 0.0, 2.0, 0.5, 0);
        set(b + 1, 0.0, 2.0, 0.5, 0);
        set(b + 2, 0.0, 1.0, 1.0, 0);
        set(b + 3, 0.0, 2.0, 0.5, 0);
        set(b + 4, 0.1, 6.0, 1.0, 0);
    }
    for (int l = 0; l < 2; ++l) {
        const int b = 32 + 8 * l;
        set(b + 0, 0.0, 20.0, 0.25, 0);
        set(b + 1, -10.0, 10.0, 0.5, 1);
        set(b + 2, -0.5, 0.5, 1.0, 0);
        for (int i = 0; i < 5; ++i) set(b + 3 + i, 0.0, 1.0, 1.0, 0);
    }
    for (int i = 48; i < 68; ++i) set(i, 0.0, 1.0, 1.0, 0);
    for (int v = 0; v < 2; ++v) {
        const int b = 68 + 3 * v;
        set(b + 0, -24.0, 24.0, 1.0, 1);
        set(b + 1, -96.0, 96.0, 0.2, 1);
        set(b + 2, -0.5, 0.5, 1.0, 0);
    }
    for (int i = 74; i < 78; ++i) set(i, 0.0, 1.0, 1.0, 0);
}

int check_nebula(const ts_range *t) {
    for (int i = 0; i < TS_NPARAM; ++i) {
        const ts_range &r = t[i];
        if (!(r.curve > 0.0) || !isfinite(r.lo) || !isfinite(r.hi) || !isfinite(r.curve))
            return fail(TS_EINVAL, "nebula entries must be finite with curve > 0%s");
        // weights (LFO shapes 35..39, 43..47; modulation mixer 48..67) are normalised by their sum: a negative
        // range would make w / sum(w), and with it the pitch, unbounded
        const bool weight = (i >= 35 && i <= 39) || (i >= 43 && i <= 47) || (i >= 48 && i <= 67);
        if (weight && (r.lo < 0.0 || r.hi < 0.0)) return fail(TS_EINVAL, "nebula ranges of weights must not be negative%s");
    }
    return TS_OK;
}

void ensure_nebula() {
    if (!S.nebula_init) {
        default_nebula(S.nebula);
        S.nebula_init = true;
        S.nebula_dirty = true;
    }
}

// The audio kernel reads frac(phase) out of the fp64 mantissa after adding 1.5*2^19, which needs the
// phase advance over one control interval to stay below 2^18 cycles (1.5*2^19 +- 2^18 keeps its exponent).
// ts_set_nebula keeps the weight rows non-negative, so |M_d| <= 1 and pitch <= midi + tune + |depth|.
bool nebula_supported(int sr) {
    const ts_range *n = S.nebula;
    auto hi = [&](int i) { return fmax(n[i].lo, n[i].hi); };
    auto mag = [&](int i) { return fmax(fabs(n[i].lo), fabs(n[i].hi)); };
    const double p1 = hi(0) + hi(68) + mag(69), p2 = hi(0) + hi(71) + mag(72);
    const double inc = (440.0 / sr) * exp2((fmax(p1, p2) - 69.0) / 12.0);
    return inc * TS_R < 262000.0;
}

// Does the active nebula leave a long exactly-silent tail in a buffer of `seconds`?  Every voice is silent after
// duration + the longest release of the four audible envelopes (H6); if even the longest such voice leaves a fifth of
// the buffer silent, the audio kernel lets its audible CTAs write the tails (ts_audio.cu, TAIL = 1).
double nebula_t_end() {  // no voice of the active nebula is audible after this time (u is clamped to [0,1], S3)
    const ts_range *n = S.nebula;
    auto hi = [&](int i) { return fmax(n[i].lo, n[i].hi); };
    return hi(1) + fmax(fmax(hi(5), hi(10)), fmax(hi(15), hi(25)));
}
int tails_expected(double seconds) { return nebula_t_end() < 0.8 * seconds; }
// Upper bound of n_act over all voices (samples): the setup kernel's first silent tick is the first j with
// j R / sr - D >= rl_max, so j <= ceil(t_end sr / R) (+1 tick against the rounding of the division); the audio kernel
// launches no CTAs for tiles that cannot be audible.
int64_t max_audible_samples(int sr, int64_t N) {
    const double ticks = ceil(nebula_t_end() * (double)sr / (double)TS_R) + 1.0;
    const double n = ticks * (double)TS_R;
    return (n < (double)N) ? (int64_t)n : N;
}

int chunk_voices(int B, int K) {
    size_t per = (size_t)K * sizeof(ts_tick);
    size_t c = TS_TABLE_BUDGET / per;
    if (c < 1) c = 1;
    if (c > (size_t)B) c = (size_t)B;
    const size_t n = ((size_t)B + c - 1) / c;  // chunks needed; spread the voices evenly over them
    return (int)(((size_t)B + n - 1) / n);
}
struct ws_layout_t {
    size_t off_hdr, off_vc, off_agg, agg_bytes, total;
};
ws_layout_t ws_layout(int Bc, int K, bool table) {
    auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
    ws_layout_t L;
    L.off_hdr = table ? up((size_t)Bc * K * sizeof(ts_tick)) : 0;
    L.off_vc = L.off_hdr + up((size_t)Bc * sizeof(ts_vhdr));
    L.off_agg = L.off_vc + up((size_t)Bc * sizeof(ts_voice_consts));
    L.agg_bytes = ts_control_agg_bytes(Bc, K);
    L.total = L.off_agg + up(L.agg_bytes);
    return L;
}

// Grows the workspace if needed and makes sure the look-back slots of THIS layout hold no flag a future epoch could
// equal: the slots sit at an offset that depends on (Bc, K), so after a layout change they alias bytes that held
// table or header data; they are cleared and the epoch count restarts whenever the layout changes.
int ensure_ws(const ws_layout_t &L, int Bc, int K) {
    ts_lane &ln = *S.cur;
    if (L.total > ln.ws_bytes) {
        if (ln.ws) {
            cudaStreamSynchronize(ln.stream);
            if (ln.audio_stream) cudaStreamSynchronize(ln.audio_stream);
            cudaFree(ln.ws);
        }
        ln.ws = nullptr;
        ln.ws_bytes = 0;
        ln.aud_pending = false;
        if (cudaMalloc(&ln.ws, L.total) != cudaSuccess) {
            cudaGetLastError();
            return fail(TS_ENOMEM, "workspace allocation failed%s");
        }
        ln.ws_bytes = L.total;
        ln.lay_B = ln.lay_K = 0;
    }
    if (ln.lay_B != Bc || ln.lay_K != K || ln.lay_off != L.off_agg) {
        if (ln.aud_pending) {  // an audio kernel may still read the old layout's table
            TS_CUDA(cudaStreamWaitEvent(ln.stream, ln.aud_done, 0));
            ln.aud_pending = false;
        }
        TS_CUDA(cudaMemsetAsync(static_cast<char *>(ln.ws) + L.off_agg, 0, L.agg_bytes, ln.stream));
        ln.epoch = 0;
        ln.lay_B = Bc;
        ln.lay_K = K;
        ln.lay_off = L.off_agg;
    }
    return TS_OK;
}

int check_sizes(int B, int sr, double seconds, int64_t *N, int *K, int R = TS_R) {
    if (B <= 0 || sr <= 0 || !(seconds > 0.0) || R <= 0) return fail(TS_EINVAL, "B, sr, seconds and R must be positive%s");
    const double ns = (double)sr * seconds;
    if (!(ns < 2.0e9)) return fail(TS_EINVAL, "sr*seconds too large%s");
    *N = ts_num_samples(sr, seconds);
    if (*N <= 0) return fail(TS_EINVAL, "zero samples%s");
    *K = (int)ts_num_ticks_r(*N, R);
    if ((double)B * (double)*N > 9.0e18 / 8) return fail(TS_EINVAL, "B*N overflows%s");
    return TS_OK;
}

int prepare_common(int sr) {
    ensure_nebula();
    if (!nebula_supported(sr)) return fail(TS_EINVAL, "nebula allows an oscillator increment above 2^18/R cycles per sample at this sr%s");
    if (S.nebula_dirty) {
        TS_CUDA(ts_upload_nebula(S.nebula, S.cur->stream));
        S.nebula_dirty = false;
    }
    if (!S.math_uploaded) {
        TS_CUDA(ts_upload_math_tables(S.cur->stream));
        S.math_uploaded = true;
    }
    return TS_OK;
}
int prepare_lane() {
    ts_lane &ln = *S.cur;
    if (!ln.d_active) {
        TS_CUDA(cudaMalloc(&ln.d_active, sizeof(unsigned long long)));
        TS_CUDA(cudaMallocHost(&ln.h_active, sizeof(unsigned long long)));
        *ln.h_active = 0;
        TS_CUDA(cudaMalloc(&ln.d_err, sizeof(unsigned int)));
        TS_CUDA(cudaMallocHost(&ln.h_err, sizeof(unsigned int)));
        *ln.h_err = 0;
        TS_CUDA(cudaMemsetAsync(ln.d_err, 0, sizeof(unsigned int), ln.stream));
    }
    return TS_OK;
}

struct sample_spec {  // the fused sampler of the streaming path: draw the records in the setup kernel
    bool on;
    uint64_t seed, g0;
};

// mode 0: audio (+ optional params_human); 1/2: debug phase of VCO 1/2; 3: debug controls of the audio path;
// mode 4: control-rate rendering on its own (no oscillator stage; tick spacing R); mode 5: audio with R = 1
int render_impl(ts_voice *d_params, sample_spec smp, int B, int sr, double seconds, int fmt, void *audio, float *params_human,
                int mode, double *dbg, int R = TS_R) {
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K, R);
    if (rc) return rc;
    if (!fmt_ok(fmt)) return fail(TS_EINVAL, "unknown output format%s");
    if (S.cur == &S.lane[0]) {  // the streaming calls upload on the caller's stream before they fork
        rc = prepare_common(sr);
        if (rc) return rc;
    }
    rc = prepare_lane();
    if (rc) return rc;
    const bool with_table = (mode != 4);
    int Bc = with_table ? chunk_voices(B, K) : B;
    if (!with_table) {  // control-rate rendering: bound the look-back slots and the per-launch grid
        const size_t cap = ((size_t)1 << 25) / (size_t)K;
        if ((size_t)Bc > cap) Bc = cap ? (int)cap : 1;
    }
    const ws_layout_t L = ws_layout(Bc, K, with_table);
    rc = ensure_ws(L, Bc, K);
    if (rc) return rc;
    ts_lane &ln = *S.cur;
    char *ws = static_cast<char *>(ln.ws);
    ts_tick *table = reinterpret_cast<ts_tick *>(ws);
    ts_vhdr *hdr = reinterpret_cast<ts_vhdr *>(ws + L.off_hdr);
    ts_voice_consts *vc = reinterpret_cast<ts_voice_consts *>(ws + L.off_vc);
    void *agg = ws + L.off_agg;
    const size_t es = fmt_bytes(fmt);

    if (S.timing && mode == 0)
        for (auto &e : S.ev)
            if (!e) TS_CUDA(cudaEventCreate(&e));
    S.ms[0] = S.ms[1] = 0.f;
    int64_t launches = 0, chunks = 0;
    const bool want_stats = S.timing;  // the active-sample count costs a memset and a copy per call
    if (want_stats) TS_CUDA(cudaMemsetAsync(ln.d_active, 0, sizeof(unsigned long long), ln.stream));

    for (int b0 = 0; b0 < B; b0 += Bc) {
        const int nb = (B - b0 < Bc) ? (B - b0) : Bc;
        const bool timed = S.timing && mode == 0;
        if (timed) TS_CUDA(cudaEventRecord(S.ev[0], ln.stream));
        if (ln.aud_pending) {  // the audio kernel still reading this workspace's table goes first
            TS_CUDA(cudaStreamWaitEvent(ln.stream, ln.aud_done, 0));
            ln.aud_pending = false;
        }
        if (++ln.epoch == 0) {  // wrapped after 2^32 launches: clear the flags and start over
            TS_CUDA(cudaMemsetAsync(agg, 0, L.agg_bytes, ln.stream));
            ln.epoch = 1;
        }
        TS_CUDA(ts_launch_setup(d_params + b0, smp.on ? 1 : 0, smp.seed, smp.g0 + (uint64_t)b0, nb, sr, R, N, K, vc, hdr,
                                params_human ? params_human + (size_t)b0 * TS_NPARAM : nullptr,
                                want_stats ? ln.d_active : nullptr, (mode == 1 || mode == 2 || mode == 3) ? 1 : 0, S.batch_table,
                                ln.stream));
        TS_CUDA(ts_launch_control(vc, nb, sr, R, N, K, table, agg, ln.epoch,
                                  (mode == 3 || mode == 4) ? dbg + (size_t)b0 * 5 * K : nullptr, with_table ? 1 : 0,
                                  (mode == 0) ? max_audible_samples(sr, N) : (int64_t)-1, ln.d_err,
                                  ln.stream));
        launches += 2;
        if (timed) TS_CUDA(cudaEventRecord(S.ev[1], ln.stream));
        cudaStream_t ast = ln.stream;
        if (ln.audio_stream && mode == 0) {  // hand over to the audio stream
            ast = ln.audio_stream;
            TS_CUDA(cudaEventRecord(ln.ctl_done, ln.stream));
            TS_CUDA(cudaStreamWaitEvent(ast, ln.ctl_done, 0));
        }
        if (mode == 5) {
            TS_CUDA(ts_launch_audio_r1(table, hdr, nb, N, K, static_cast<float *>(audio) + (size_t)b0 * N, ast));
            ++launches;
        } else if (mode <= 2) {
            TS_CUDA(ts_launch_audio(table, hdr, nb, N, K, audio ? static_cast<char *>(audio) + (size_t)b0 * N * es : nullptr, fmt,
                                    mode, tails_expected(seconds), max_audible_samples(sr, N),
                                    (mode == 1 || mode == 2) ? dbg + (size_t)b0 * N : nullptr, ast));
            ++launches;
        }
        if (ast != ln.stream) {  // the next control launch on this workspace will wait for this audio kernel
            TS_CUDA(cudaEventRecord(ln.aud_done, ast));
            ln.aud_pending = true;
        }
        if (timed) {
            TS_CUDA(cudaEventRecord(S.ev[2], ln.stream));
            TS_CUDA(cudaEventSynchronize(S.ev[2]));
            float a = 0.f, b = 0.f;
            TS_CUDA(cudaEventElapsedTime(&a, S.ev[0], S.ev[1]));
            TS_CUDA(cudaEventElapsedTime(&b, S.ev[1], S.ev[2]));
            S.ms[0] += a;
            S.ms[1] += b;
        }
        ++chunks;
    }
    if (want_stats)
        TS_CUDA(cudaMemcpyAsync(ln.h_active, ln.d_active, sizeof(unsigned long long), cudaMemcpyDeviceToHost, ln.stream));
    S.stats[0] = launches;
    S.stats[1] = chunks;
    return TS_OK;
}

int ensure_streams() {
    if (S.fork) return TS_OK;
    int lo_p = 0, hi_p = 0;
    TS_CUDA(cudaDeviceGetStreamPriorityRange(&lo_p, &hi_p));  // numerically lower = higher priority
    for (int x = 0; x < TS_SL; ++x) {
        TS_CUDA(cudaStreamCreateWithPriority(&S.hi[x], cudaStreamNonBlocking, hi_p));
        TS_CUDA(cudaStreamCreateWithPriority(&S.lo[x], cudaStreamNonBlocking, lo_p));
        S.lane[1 + x].stream = S.hi[x];
        S.lane[1 + x].audio_stream = S.lo[x];
        TS_CUDA(cudaEventCreateWithFlags(&S.lane[1 + x].ctl_done, cudaEventDisableTiming));
        TS_CUDA(cudaEventCreateWithFlags(&S.lane[1 + x].aud_done, cudaEventDisableTiming));
    }
    for (auto &e : S.join_ev) TS_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    for (auto &b : S.batch_done)
        for (auto &e : b) TS_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    TS_CUDA(cudaEventCreateWithFlags(&S.fork, cudaEventDisableTiming));
    return TS_OK;
}

// All internal streams start after everything already queued on the caller's stream.
int fork_streams() {
    TS_CUDA(cudaEventRecord(S.fork, S.lane[0].stream));
    for (int x = 0; x < TS_SL; ++x) {
        TS_CUDA(cudaStreamWaitEvent(S.hi[x], S.fork, 0));
        TS_CUDA(cudaStreamWaitEvent(S.lo[x], S.fork, 0));
    }
    return TS_OK;
}

// A batch on the internal streams (forked by the caller): the voice chunks of the batch rotate over the
// streaming lanes, setup + control on `hi`, audio on `lo`, so that the control stage of one chunk overlaps the audio
// stage of the previous one -- across the chunks of a batch as well as across batches.
// seq: position of the batch in its sequence (chunk j of the batch runs on lane (seq + j) % TS_SL).  n_ring > 0: the batch
// goes into the ring slot that batch seq - n_ring wrote: that batch's audio, possibly on the other audio stream, must
// have finished first.
int stream_batch(ts_voice *p, sample_spec smp, int B, int sr, double seconds, int fmt, void *a, float *params_human, uint64_t seq = 0,
                 int n_ring = 0) {
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K);
    if (rc) return rc;
    const int Bc = chunk_voices(B, K);
    // Single-chunk batches rotate strictly over the lanes; with a ring that is a multiple of TS_SL a slot is then always
    // written on the same audio stream and stream order covers the hazard.
    const bool same_stream = (Bc >= B) && (n_ring % TS_SL == 0);
    if (n_ring > 0 && !same_stream) {
        const uint64_t k = (uint64_t)(n_ring < TS_MAX_RING ? n_ring : TS_MAX_RING);
        if (seq >= k) {
            cudaEvent_t *ev = S.batch_done[(seq - k) % TS_MAX_RING];
            // lo: the slot's audio; hi: the slot's parameter records, written by the setup kernel of whichever lane the batch
            // runs on (the old batch's audio finished => its setup kernel, which the audio waited for, finished too)
            for (int x = 0; x < TS_SL; ++x)
                for (int y = 0; y < TS_SL; ++y) {
                    TS_CUDA(cudaStreamWaitEvent(S.lo[x], ev[y], 0));
                    TS_CUDA(cudaStreamWaitEvent(S.hi[x], ev[y], 0));
                }
        }
    }
    const size_t es = fmt_bytes(fmt);
    const bool timing = S.timing;
    S.timing = false;  // per-kernel events would serialise the streams
    int64_t launches = 0, chunks = 0;
    for (int b0 = 0; b0 < B && rc == TS_OK; b0 += Bc) {
        const int nb = (B - b0 < Bc) ? (B - b0) : Bc;
        S.cur = &S.lane[1 + (int)((seq + (uint64_t)chunks) % (uint64_t)TS_SL)];
        rc = render_impl(p + b0, sample_spec{smp.on, smp.seed, smp.g0 + (uint64_t)b0}, nb, sr, seconds, fmt,
                         static_cast<char *>(a) + (size_t)b0 * (size_t)N * es,
                         params_human ? params_human + (size_t)b0 * TS_NPARAM : nullptr, 0, nullptr);
        launches += S.stats[0];
        ++chunks;
    }
    S.timing = timing;
    S.cur = &S.lane[0];
    S.stats[0] = launches;
    S.stats[1] = chunks;
    if (rc == TS_OK && n_ring > 0 && !same_stream)
        for (int x = 0; x < TS_SL; ++x) TS_CUDA(cudaEventRecord(S.batch_done[seq % TS_MAX_RING][x], S.lo[x]));
    return rc;
}

// The caller's stream continues after all internal streams.
int join_streams() {
    for (int x = 0; x < TS_SL; ++x) {
        TS_CUDA(cudaEventRecord(S.join_ev[2 * x], S.hi[x]));
        TS_CUDA(cudaStreamWaitEvent(S.lane[0].stream, S.join_ev[2 * x], 0));
        TS_CUDA(cudaEventRecord(S.join_ev[2 * x + 1], S.lo[x]));
        TS_CUDA(cudaStreamWaitEvent(S.lane[0].stream, S.join_ev[2 * x + 1], 0));
    }
    return TS_OK;
}

int corpus_issue(uint64_t batch) {  // render `batch` into its slot and record the slot's ready event on `lo`
    ts_corpus_state &C = S.corpus;
    const int slot = (int)(batch % (uint64_t)C.cfg.n_ring);
    const size_t es = fmt_bytes(C.cfg.fmt);
    const int rc = stream_batch(C.cfg.d_params_ring + (size_t)slot * (size_t)C.cfg.B,
                                sample_spec{true, C.cfg.seed, batch * (uint64_t)C.cfg.B}, C.cfg.B, C.cfg.sr, C.cfg.seconds, C.cfg.fmt,
                                static_cast<char *>(C.cfg.d_audio_ring) + (size_t)slot * (size_t)C.cfg.B * (size_t)C.N * es, nullptr,
                                batch - C.first, C.cfg.n_ring);
    if (rc) return rc;
    // the slot is ready when the batch's audio on BOTH audio streams has finished
    for (int x = 1; x < TS_SL; ++x) {
        TS_CUDA(cudaEventRecord(S.join_ev[2 * x + 1], S.lo[x]));
        TS_CUDA(cudaStreamWaitEvent(S.lo[0], S.join_ev[2 * x + 1], 0));
    }
    TS_CUDA(cudaEventRecord(C.ready[slot], S.lo[0]));
    return TS_OK;
}

// A batch that needs several voice chunks (control table capped for L2) runs its chunks on the internal lanes, so
// that setup + control of chunk k+1 overlap the audio kernel of chunk k; a single-chunk batch stays on the set stream.
int render_audio(ts_voice *d_params, sample_spec smp, int B, int sr, double seconds, int fmt, void *d_audio, float *d_params_human) {
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K);
    if (rc) return rc;
    if (chunk_voices(B, K) >= B || S.timing || S.corpus.open)
        return render_impl(d_params, smp, B, sr, seconds, fmt, d_audio, d_params_human, 0, nullptr);
    if (!fmt_ok(fmt)) return fail(TS_EINVAL, "unknown output format%s");
    S.cur = &S.lane[0];
    rc = prepare_common(sr);
    if (rc) return rc;
    rc = ensure_streams();
    if (rc) return rc;
    rc = fork_streams();
    if (rc) return rc;
    rc = stream_batch(d_params, smp, B, sr, seconds, fmt, d_audio, d_params_human);
    const int rj = join_streams();
    return rc ? rc : rj;
}

}  // namespace

extern "C" {

int ts_corpus_is_test(uint64_t g) { return (g / 1024u) % 10u == 9u; }

int64_t ts_num_samples(int sr, double seconds) { return (int64_t)llround((double)sr * seconds); }
int64_t ts_num_ticks(int64_t N) { return (N + TS_R - 1) / TS_R + 1; }
int ts_streaming_lanes(void) { return TS_SL; }
int64_t ts_num_ticks_r(int64_t N, int R) { return (R > 0) ? (N + R - 1) / R + 1 : 0; }

int ts_sample_params(uint64_t seed, uint64_t batch_index, int B, ts_voice *d_params) {
    if (!d_params) return fail(TS_ENULL, "d_params is NULL%s");
    if (B <= 0) return fail(TS_EINVAL, "B must be positive%s");
    TS_CUDA(ts_launch_sample(seed, batch_index * (uint64_t)B, B, d_params, S.cur->stream));
    return TS_OK;
}

int ts_render_fmt(const ts_voice *d_params, int B, int sr, double seconds, int fmt, void *d_audio, float *d_params_human) {
    if (!d_params) return fail(TS_ENULL, "d_params is NULL%s");
    if (!d_audio) return fail(TS_ENULL, "audio is NULL%s");
    return render_audio(const_cast<ts_voice *>(d_params), sample_spec{false, 0, 0}, B, sr, seconds, fmt, d_audio, d_params_human);
}

int ts_render(const ts_voice *d_params, int B, int sr, double seconds, ts_out out) {
    if (!d_params) return fail(TS_ENULL, "d_params is NULL%s");
    if (!out.audio) return fail(TS_ENULL, "out.audio is NULL%s");
    return ts_render_fmt(d_params, B, sr, seconds, TS_F32, out.audio, out.params_human);
}

int ts_render_host_fmt(uint64_t seed, uint64_t batch_index, int B, int sr, double seconds, int fmt, void *host_audio,
                       ts_voice *host_params) {
    if (!host_audio) return fail(TS_ENULL, "host_audio is NULL%s");
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K);
    if (rc) return rc;
    if (!fmt_ok(fmt)) return fail(TS_EINVAL, "unknown output format%s");
    const size_t pbytes = ((size_t)B * sizeof(ts_voice) + 255) & ~(size_t)255;
    const size_t abytes = (size_t)B * N * fmt_bytes(fmt);
    if (pbytes + abytes > S.stage_bytes) {
        if (S.stage) cudaFree(S.stage);
        S.stage = nullptr;
        S.stage_bytes = 0;
        if (cudaMalloc(&S.stage, pbytes + abytes) != cudaSuccess) {
            cudaGetLastError();
            return fail(TS_ENOMEM, "staging allocation failed%s");
        }
        S.stage_bytes = pbytes + abytes;
    }
    ts_voice *d_params = static_cast<ts_voice *>(S.stage);
    void *d_audio = static_cast<char *>(S.stage) + pbytes;
    rc = render_audio(d_params, sample_spec{true, seed, batch_index * (uint64_t)B}, B, sr, seconds, fmt, d_audio, nullptr);
    if (rc) return rc;
    TS_CUDA(cudaMemcpyAsync(host_audio, d_audio, abytes, cudaMemcpyDeviceToHost, S.cur->stream));
    if (host_params)
        TS_CUDA(cudaMemcpyAsync(host_params, d_params, (size_t)B * sizeof(ts_voice), cudaMemcpyDeviceToHost, S.cur->stream));
    return ts_sync();
}

int ts_render_host(uint64_t seed, uint64_t batch_index, int B, int sr, double seconds, float *host_audio,
                   ts_voice *host_params) {
    return ts_render_host_fmt(seed, batch_index, B, sr, seconds, TS_F32, host_audio, host_params);
}

int ts_corpus_render_fmt(uint64_t seed, uint64_t first_batch, int n_batches, int B, int sr, double seconds, int fmt,
                         ts_voice *d_params_ring, void *d_audio_ring, int n_ring) {
    if (!d_params_ring || !d_audio_ring) return fail(TS_ENULL, "NULL ring%s");
    if (n_batches <= 0 || n_ring <= 0) return fail(TS_EINVAL, "n_batches and n_ring must be positive%s");
    if (S.corpus.open) return fail(TS_EINVAL, "a corpus iterator is open: close it first%s");
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K);
    if (rc) return rc;
    if (!fmt_ok(fmt)) return fail(TS_EINVAL, "unknown output format%s");
    S.cur = &S.lane[0];
    rc = prepare_common(sr);  // nebula / tables go up on the caller's stream, before the fork
    if (rc) return rc;
    rc = ensure_streams();
    if (rc) return rc;
    rc = fork_streams();
    if (rc) return rc;
    // Ring hazards: a slot's records are written by the setup kernel (a `hi` stream) and its audio by the audio kernel (a
    // `lo` stream) of the lane the batch runs on.  A single-chunk batch in a ring that is a multiple of the lanes always
    // meets its slot on the same pair of streams (stream order covers it); otherwise stream_batch makes every internal
    // stream wait for the audio of the batch that used the slot before.
    const size_t es = fmt_bytes(fmt);
    int64_t launches = 0;
    for (int i = 0; i < n_batches && rc == TS_OK; ++i) {
        const size_t slot = (size_t)(i % n_ring);
        rc = stream_batch(d_params_ring + slot * (size_t)B, sample_spec{true, seed, (first_batch + (uint64_t)i) * (uint64_t)B}, B, sr,
                          seconds, fmt, static_cast<char *>(d_audio_ring) + slot * (size_t)B * (size_t)N * es, nullptr, (uint64_t)i, n_ring);
        launches += S.stats[0];
    }
    const int rj = join_streams();
    S.stats[0] = launches;  // kernels launched by this call (3 per batch and voice chunk)
    return rc ? rc : rj;
}

int ts_corpus_render(uint64_t seed, uint64_t first_batch, int n_batches, int B, int sr, double seconds,
                     ts_voice *d_params_ring, float *d_audio_ring, int n_ring) {
    return ts_corpus_render_fmt(seed, first_batch, n_batches, B, sr, seconds, TS_F32, d_params_ring, d_audio_ring, n_ring);
}

int ts_corpus_render_nebulae(uint64_t seed, uint64_t first_batch, int n_batches, int B, int sr, double seconds, int fmt,
                             const ts_range *host_tables, ts_voice *d_params_ring, void *d_audio_ring, int n_ring) {
    if (!host_tables) return fail(TS_ENULL, "host_tables is NULL%s");
    if (!d_params_ring || !d_audio_ring) return fail(TS_ENULL, "NULL ring%s");
    if (n_batches <= 0 || n_ring <= 0) return fail(TS_EINVAL, "n_batches and n_ring must be positive%s");
    if (S.corpus.open) return fail(TS_EINVAL, "a corpus iterator is open: close it first%s");
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K);
    if (rc) return rc;
    if (!fmt_ok(fmt)) return fail(TS_EINVAL, "unknown output format%s");
    ensure_nebula();
    ts_range saved[TS_NPARAM];
    memcpy(saved, S.nebula, sizeof saved);
    // every table is checked before anything is launched (a refused table leaves nothing half rendered)
    for (int i = 0; i < n_batches; ++i) {
        rc = check_nebula(host_tables + (size_t)i * TS_NPARAM);
        if (rc) return rc;
        memcpy(S.nebula, host_tables + (size_t)i * TS_NPARAM, sizeof S.nebula);
        const bool ok = nebula_supported(sr);
        memcpy(S.nebula, saved, sizeof saved);
        if (!ok) return fail(TS_EINVAL, "a table allows an oscillator increment above 2^18/R cycles per sample at this sr%s");
    }
    S.cur = &S.lane[0];
    rc = prepare_common(sr);  // math tables (and the active nebula, if stale) go up on the caller's stream, before the fork
    if (rc) return rc;
    rc = ensure_streams();
    if (rc) return rc;
    // all tables of the call, in the device layout, in one upload on the caller's stream
    const size_t tb = ts_nebula_device_bytes(), need = tb * (size_t)n_batches;
    if (!S.tables_up) TS_CUDA(cudaEventCreateWithFlags(&S.tables_up, cudaEventDisableTiming));
    else TS_CUDA(cudaEventSynchronize(S.tables_up));  // the previous call's upload has read the pinned staging buffer
    if (need > S.tables_bytes) {
        TS_CUDA(cudaStreamSynchronize(S.lane[0].stream));  // kernels of an earlier call may still read the old device copy
        if (S.d_tables) cudaFree(S.d_tables);
        if (S.h_tables) cudaFreeHost(S.h_tables);
        S.d_tables = S.h_tables = nullptr;
        S.tables_bytes = 0;
        if (cudaMalloc(&S.d_tables, need) != cudaSuccess || cudaMallocHost(&S.h_tables, need) != cudaSuccess) {
            cudaGetLastError();
            return fail(TS_ENOMEM, "allocation of the nebula tables failed%s");
        }
        S.tables_bytes = need;
    }
    for (int i = 0; i < n_batches; ++i)
        ts_nebula_to_device_layout(host_tables + (size_t)i * TS_NPARAM, static_cast<char *>(S.h_tables) + tb * (size_t)i);
    TS_CUDA(cudaMemcpyAsync(S.d_tables, S.h_tables, need, cudaMemcpyHostToDevice, S.lane[0].stream));
    TS_CUDA(cudaEventRecord(S.tables_up, S.lane[0].stream));
    rc = fork_streams();
    if (rc) return rc;
    const size_t es = fmt_bytes(fmt);
    int64_t launches = 0;
    for (int i = 0; i < n_batches && rc == TS_OK; ++i) {
        const size_t slot = (size_t)(i % n_ring);
        // the host-side decisions of a batch (silent-tail mode, launch extents) follow the batch's own table
        memcpy(S.nebula, host_tables + (size_t)i * TS_NPARAM, sizeof S.nebula);
        S.batch_table = static_cast<const char *>(S.d_tables) + tb * (size_t)i;
        rc = stream_batch(d_params_ring + slot * (size_t)B, sample_spec{true, seed, (first_batch + (uint64_t)i) * (uint64_t)B}, B, sr,
                          seconds, fmt, static_cast<char *>(d_audio_ring) + slot * (size_t)B * (size_t)N * es, nullptr, (uint64_t)i, n_ring);
        launches += S.stats[0];
    }
    S.batch_table = nullptr;
    memcpy(S.nebula, saved, sizeof saved);  // the active nebula is what it was
    const int rj = join_streams();
    S.stats[0] = launches;
    return rc ? rc : rj;
}

// A batch could not be issued (TS_ENOMEM, TS_ECUDA): the iterator does not stay half open with batches in flight -- the
// internal streams are drained, the iterator is closed and the first error (code and text) is what the caller sees.
static int corpus_abort(int rc) {
    char first[sizeof S.err];
    memcpy(first, S.err, sizeof first);
    ts_corpus_close();
    memcpy(S.err, first, sizeof first);
    return rc;
}

int ts_corpus_open(const ts_corpus_cfg *host_cfg, uint64_t first_batch) {
    if (!host_cfg) return fail(TS_ENULL, "host_cfg is NULL%s");
    if (!host_cfg->d_audio_ring || !host_cfg->d_params_ring) return fail(TS_ENULL, "NULL ring%s");
    if (host_cfg->n_ring < 2 || host_cfg->n_ring > TS_MAX_RING) return fail(TS_EINVAL, "n_ring must be in [2, 64]%s");
    if (S.corpus.open) return fail(TS_EINVAL, "a corpus iterator is already open%s");
    int64_t N;
    int K;
    int rc = check_sizes(host_cfg->B, host_cfg->sr, host_cfg->seconds, &N, &K);
    if (rc) return rc;
    if (!fmt_ok(host_cfg->fmt)) return fail(TS_EINVAL, "unknown output format%s");
    S.cur = &S.lane[0];
    rc = prepare_common(host_cfg->sr);
    if (rc) return rc;
    rc = ensure_streams();
    if (rc) return rc;
    ts_corpus_state &C = S.corpus;
    C.cfg = *host_cfg;
    C.N = N;
    C.first = C.next_out = C.next_render = first_batch;
    for (int i = 0; i < host_cfg->n_ring; ++i)
        if (!C.ready[i]) TS_CUDA(cudaEventCreateWithFlags(&C.ready[i], cudaEventDisableTiming));
    if (!C.consumed) TS_CUDA(cudaEventCreateWithFlags(&C.consumed, cudaEventDisableTiming));
    rc = fork_streams();
    if (rc) return rc;
    C.open = true;
    for (int i = 0; i < host_cfg->n_ring - 1; ++i) {  // render ahead: every slot but one
        rc = corpus_issue(C.next_render++);
        if (rc) return corpus_abort(rc);
    }
    return TS_OK;
}

int ts_corpus_next(ts_corpus_batch *host_out) {
    if (!host_out) return fail(TS_ENULL, "host_out is NULL%s");
    ts_corpus_state &C = S.corpus;
    if (!C.open) return fail(TS_EINVAL, "no corpus iterator is open%s");
    // The slot handed out by the previous call is free once the caller's stream reaches this point, and it is the one
    // slot not in flight: the batch n_ring - 1 ahead of the one handed out now goes into it, ordered after the caller's
    // stream (both internal streams wait for it).
    TS_CUDA(cudaEventRecord(C.consumed, S.lane[0].stream));
    for (int x = 0; x < TS_SL; ++x) {
        TS_CUDA(cudaStreamWaitEvent(S.lo[x], C.consumed, 0));
        TS_CUDA(cudaStreamWaitEvent(S.hi[x], C.consumed, 0));
    }
    const int rc = corpus_issue(C.next_render++);
    if (rc) return corpus_abort(rc);
    const uint64_t b = C.next_out++;
    const int slot = (int)(b % (uint64_t)C.cfg.n_ring);
    TS_CUDA(cudaStreamWaitEvent(S.lane[0].stream, C.ready[slot], 0));  // the caller's stream waits for this batch
    host_out->d_audio = static_cast<char *>(C.cfg.d_audio_ring) + (size_t)slot * (size_t)C.cfg.B * (size_t)C.N * fmt_bytes(C.cfg.fmt);
    host_out->d_params = C.cfg.d_params_ring + (size_t)slot * (size_t)C.cfg.B;
    host_out->batch_index = b;
    host_out->first_voice = b * (uint64_t)C.cfg.B;
    host_out->is_test_first = ts_corpus_is_test(host_out->first_voice);
    host_out->is_test_last = ts_corpus_is_test(host_out->first_voice + (uint64_t)C.cfg.B - 1);
    host_out->slot = slot;
    return TS_OK;
}

int ts_corpus_close(void) {
    ts_corpus_state &C = S.corpus;
    if (!C.open) return TS_OK;
    C.open = false;
    for (int x = 0; x < TS_SL; ++x) {
        TS_CUDA(cudaStreamSynchronize(S.hi[x]));
        TS_CUDA(cudaStreamSynchronize(S.lo[x]));
    }
    return TS_OK;
}

int ts_set_stream(void *cuda_stream) {
    S.lane[0].stream = static_cast<cudaStream_t>(cuda_stream);
    return TS_OK;
}

int ts_default_nebula(ts_range host_out78[TS_NPARAM]) {
    if (!host_out78) return fail(TS_ENULL, "host_out78 is NULL%s");
    default_nebula(host_out78);
    return TS_OK;
}

int ts_set_nebula(const ts_range *host_in78) {
    // The iterator's batches are issued without re-uploading the table (corpus_issue -> render_impl on the streaming lanes),
    // so a change here would split the device table from the host-side extent / silent-tail decisions, and a later
    // ts_render would upload over a table the iterator's setup kernels are still reading.
    if (S.corpus.open) return fail(TS_EINVAL, "a corpus iterator is open (its nebula is fixed at ts_corpus_open): close it first%s");
    if (!host_in78) {
        default_nebula(S.nebula);
    } else {
        const int rc = check_nebula(host_in78);
        if (rc) return rc;
        memcpy(S.nebula, host_in78, sizeof S.nebula);
    }
    S.nebula_init = true;
    S.nebula_dirty = true;
    return TS_OK;
}

size_t ts_workspace_bytes(int B, int sr, double seconds) {
    int64_t N;
    int K;
    if (check_sizes(B, sr, seconds, &N, &K)) return 0;
    return ws_layout(chunk_voices(B, K), K, true).total;
}

const char *ts_last_error(void) { return S.err; }

int ts_sync(void) {
    ts_lane &ln = S.lane[0];
    // the error flags of all lanes (the streaming calls join the set stream before they return)
    for (int l = 0; l < TS_LANES; ++l)
        if (S.lane[l].d_err)
            TS_CUDA(cudaMemcpyAsync(S.lane[l].h_err, S.lane[l].d_err, sizeof(unsigned int), cudaMemcpyDeviceToHost, ln.stream));
    TS_CUDA(cudaStreamSynchronize(ln.stream));
    if (ln.h_active) S.stats[2] = (int64_t)*ln.h_active;
    bool bad = false;
    for (int l = 0; l < TS_LANES; ++l)
        if (S.lane[l].h_err && *S.lane[l].h_err) {
            bad = true;
            *S.lane[l].h_err = 0;
            cudaMemsetAsync(S.lane[l].d_err, 0, sizeof(unsigned int), ln.stream);
        }
    if (bad) return fail(TS_ECUDA, "a control kernel gave up waiting for a predecessor chunk (look-back timeout)%s");
    return TS_OK;
}

void ts_shutdown(void) {
    if (S.corpus.open) ts_corpus_close();
    for (auto &e : S.corpus.ready)
        if (e) { cudaEventDestroy(e); e = nullptr; }
    if (S.corpus.consumed) { cudaEventDestroy(S.corpus.consumed); S.corpus.consumed = nullptr; }
    for (int l = 0; l < TS_LANES; ++l) {
        ts_lane &L = S.lane[l];
        if (L.ws) cudaFree(L.ws);
        if (L.d_active) cudaFree(L.d_active);
        if (L.h_active) cudaFreeHost(L.h_active);
        if (L.d_err) cudaFree(L.d_err);
        if (L.h_err) cudaFreeHost(L.h_err);
        if (L.ctl_done) cudaEventDestroy(L.ctl_done);
        if (L.aud_done) cudaEventDestroy(L.aud_done);
        const cudaStream_t keep = (l == 0) ? L.stream : nullptr;
        L = ts_lane();
        L.stream = keep;
    }
    if (S.fork) { cudaEventDestroy(S.fork); S.fork = nullptr; }
    for (int x = 0; x < TS_SL; ++x) {
        if (S.hi[x]) { cudaStreamDestroy(S.hi[x]); S.hi[x] = nullptr; }
        if (S.lo[x]) { cudaStreamDestroy(S.lo[x]); S.lo[x] = nullptr; }
    }
    for (auto &e : S.join_ev)
        if (e) { cudaEventDestroy(e); e = nullptr; }
    for (auto &b : S.batch_done)
        for (auto &e : b)
            if (e) { cudaEventDestroy(e); e = nullptr; }
    if (S.stage) cudaFree(S.stage);
    if (S.mmd_ws) cudaFree(S.mmd_ws);
    if (S.d_tables) cudaFree(S.d_tables);
    if (S.h_tables) cudaFreeHost(S.h_tables);
    if (S.tables_up) cudaEventDestroy(S.tables_up);
    S.d_tables = S.h_tables = nullptr;
    S.tables_bytes = 0;
    S.tables_up = nullptr;
    S.batch_table = nullptr;
    for (auto &e : S.ev)
        if (e) { cudaEventDestroy(e); e = nullptr; }
    S.stage = nullptr;
    S.stage_bytes = 0;
    S.mmd_ws = nullptr;
    S.mmd_ws_count = 0;
    S.cur = &S.lane[0];
    S.nebula_dirty = true;
    S.math_uploaded = false;
}

#ifdef TS_MEASURE  // the measurement aids of include/tsynth_measure.h: only in libtsynth_measure.so
int ts_time_kernels(const ts_voice *d_params, int B, int sr, double seconds, float *d_audio_ring, int n_ring, int reps,
                    float host_ms[2]) {
    if (!d_params || !d_audio_ring || !host_ms) return fail(TS_ENULL, "NULL argument%s");
    if (n_ring <= 0 || reps <= 0) return fail(TS_EINVAL, "n_ring and reps must be positive%s");
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K);
    if (rc) return rc;
    S.cur = &S.lane[0];
    rc = prepare_common(sr);
    if (rc) return rc;
    rc = prepare_lane();
    if (rc) return rc;
    const int Bc = chunk_voices(B, K);
    const ws_layout_t L = ws_layout(Bc, K, true);
    rc = ensure_ws(L, Bc, K);
    if (rc) return rc;
    ts_lane &ln = *S.cur;
    char *ws = static_cast<char *>(ln.ws);
    ts_tick *table = reinterpret_cast<ts_tick *>(ws);
    ts_vhdr *hdr = reinterpret_cast<ts_vhdr *>(ws + L.off_hdr);
    ts_voice_consts *vc = reinterpret_cast<ts_voice_consts *>(ws + L.off_vc);
    void *agg = ws + L.off_agg;
    for (auto &e : S.ev)
        if (!e) TS_CUDA(cudaEventCreate(&e));
    cudaStream_t st = ln.stream;
    const int tails = tails_expected(seconds);
    float a = 0.f, b = 0.f;
    for (int b0 = 0; b0 < B; b0 += Bc) {  // voice chunk by voice chunk, as ts_render launches them
        const int nb = (B - b0 < Bc) ? (B - b0) : Bc;
        TS_CUDA(cudaEventRecord(S.ev[0], st));
        for (int r = 0; r < reps; ++r) {
            if (++ln.epoch == 0) {
                TS_CUDA(cudaMemsetAsync(agg, 0, L.agg_bytes, st));
                ln.epoch = 1;
            }
            TS_CUDA(ts_launch_setup(const_cast<ts_voice *>(d_params) + b0, 0, 0, 0, nb, sr, TS_R, N, K, vc, hdr, nullptr, nullptr, 0, nullptr, st));
            TS_CUDA(ts_launch_control(vc, nb, sr, TS_R, N, K, table, agg, ln.epoch, nullptr, 1, max_audible_samples(sr, N), ln.d_err, st));
        }
        TS_CUDA(cudaEventRecord(S.ev[1], st));
        for (int r = 0; r < reps; ++r)
            TS_CUDA(ts_launch_audio(table, hdr, nb, N, K,
                                    d_audio_ring + (size_t)(r % n_ring) * (size_t)B * (size_t)N + (size_t)b0 * (size_t)N, TS_F32,
                                    0, tails, max_audible_samples(sr, N), nullptr, st));
        TS_CUDA(cudaEventRecord(S.ev[2], st));
        TS_CUDA(cudaEventSynchronize(S.ev[2]));
        float x = 0.f, y = 0.f;
        TS_CUDA(cudaEventElapsedTime(&x, S.ev[0], S.ev[1]));
        TS_CUDA(cudaEventElapsedTime(&y, S.ev[1], S.ev[2]));
        a += x;
        b += y;
    }
    host_ms[0] = a / (float)reps;
    host_ms[1] = b / (float)reps;
    return TS_OK;
}

int ts_time_audio_lanes(const ts_voice *d_params, int B, int sr, double seconds, float *d_audio_ring, int n_ring, int reps,
                              float *host_ms) {
    if (!d_params || !d_audio_ring || !host_ms) return fail(TS_ENULL, "NULL argument%s");
    if (n_ring <= 0 || reps <= 0) return fail(TS_EINVAL, "n_ring and reps must be positive%s");
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K);
    if (rc) return rc;
    if (chunk_voices(B, K) < B) return fail(TS_EINVAL, "the batch must fit one voice chunk%s");
    S.cur = &S.lane[0];
    rc = prepare_common(sr);
    if (rc) return rc;
    rc = prepare_lane();
    if (rc) return rc;
    rc = ensure_streams();
    if (rc) return rc;
    const ws_layout_t L = ws_layout(B, K, true);
    rc = ensure_ws(L, B, K);
    if (rc) return rc;
    ts_lane &ln = *S.cur;
    char *ws = static_cast<char *>(ln.ws);
    ts_tick *table = reinterpret_cast<ts_tick *>(ws);
    ts_vhdr *hdr = reinterpret_cast<ts_vhdr *>(ws + L.off_hdr);
    ts_voice_consts *vc = reinterpret_cast<ts_voice_consts *>(ws + L.off_vc);
    for (auto &e : S.ev)
        if (!e) TS_CUDA(cudaEventCreate(&e));
    cudaStream_t st = ln.stream;
    if (++ln.epoch == 0) {
        TS_CUDA(cudaMemsetAsync(ws + L.off_agg, 0, L.agg_bytes, st));
        ln.epoch = 1;
    }
    TS_CUDA(ts_launch_setup(const_cast<ts_voice *>(d_params), 0, 0, 0, B, sr, TS_R, N, K, vc, hdr, nullptr, nullptr, 0, nullptr, st));
    TS_CUDA(ts_launch_control(vc, B, sr, TS_R, N, K, table, ws + L.off_agg, ln.epoch, nullptr, 1, max_audible_samples(sr, N), ln.d_err, st));
    TS_CUDA(cudaEventRecord(S.ev[0], st));
    rc = fork_streams();
    if (rc) return rc;
    const int tails = tails_expected(seconds);
    for (int r = 0; r < reps; ++r)  // the table is only read: launches on the audio streams are independent
        TS_CUDA(ts_launch_audio(table, hdr, B, N, K, d_audio_ring + (size_t)(r % n_ring) * (size_t)B * (size_t)N, TS_F32, 0, tails,
                                max_audible_samples(sr, N), nullptr, S.lo[r % TS_SL]));
    rc = join_streams();
    if (rc) return rc;
    TS_CUDA(cudaEventRecord(S.ev[1], st));
    TS_CUDA(cudaEventSynchronize(S.ev[1]));
    float x = 0.f;
    TS_CUDA(cudaEventElapsedTime(&x, S.ev[0], S.ev[1]));
    *host_ms = x / (float)reps;
    return TS_OK;
}

int ts_time_fill(void *d_dst, size_t bytes, int reps, float *host_ms) {
    if (!d_dst || !host_ms) return fail(TS_ENULL, "NULL argument%s");
    if (bytes < 16 || reps <= 0) return fail(TS_EINVAL, "bytes and reps must be positive%s");
    for (auto &e : S.ev)
        if (!e) TS_CUDA(cudaEventCreate(&e));
    cudaStream_t st = S.lane[0].stream;
    TS_CUDA(ts_launch_fill(d_dst, bytes, st));
    TS_CUDA(cudaEventRecord(S.ev[0], st));
    for (int r = 0; r < reps; ++r) TS_CUDA(ts_launch_fill(d_dst, bytes, st));
    TS_CUDA(cudaEventRecord(S.ev[1], st));
    TS_CUDA(cudaEventSynchronize(S.ev[1]));
    float x = 0.f;
    TS_CUDA(cudaEventElapsedTime(&x, S.ev[0], S.ev[1]));
    *host_ms = x / (float)reps;
    return TS_OK;
}

int ts_time_alu_bound(int fastsin, int reps, double *host_samples_per_s) {
    if (!host_samples_per_s) return fail(TS_ENULL, "NULL argument%s");
    if (reps <= 0) return fail(TS_EINVAL, "reps must be positive%s");
    for (auto &e : S.ev)
        if (!e) TS_CUDA(cudaEventCreate(&e));
    cudaStream_t st = S.lane[0].stream;
    float *sink = nullptr;
    TS_CUDA(cudaMalloc(&sink, 1024 * sizeof(float)));
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    TS_CUDA(ts_launch_body_bench(fastsin, reps, sink, st));  // warm-up
    TS_CUDA(cudaEventRecord(S.ev[0], st));
    TS_CUDA(ts_launch_body_bench(fastsin, reps, sink, st));
    TS_CUDA(cudaEventRecord(S.ev[1], st));
    TS_CUDA(cudaEventSynchronize(S.ev[1]));
    float ms = 0.f;
    TS_CUDA(cudaEventElapsedTime(&ms, S.ev[0], S.ev[1]));
    cudaFree(sink);
    *host_samples_per_s = (double)sms * 1024.0 * (double)reps * TS_RUN / ((double)ms * 1e-3);
    return TS_OK;
}

int ts_time_pipes(double host_rates[8]) {
    if (!host_rates) return fail(TS_ENULL, "NULL argument%s");
    TS_CUDA(ts_measure_pipes(host_rates, S.lane[0].stream));
    return TS_OK;
}
#endif  // TS_MEASURE

int ts_set_timing(int enable) {
    S.timing = enable != 0;
    return TS_OK;
}
int ts_last_kernel_ms(float host_ms[2]) {
    if (!host_ms) return fail(TS_ENULL, "host_ms is NULL%s");
    host_ms[0] = S.ms[0];
    host_ms[1] = S.ms[1];
    return TS_OK;
}
int ts_last_stats(int64_t host_stats[3]) {
    if (!host_stats) return fail(TS_ENULL, "host_stats is NULL%s");
    if (S.lane[0].h_active) S.stats[2] = (int64_t)*S.lane[0].h_active;
    memcpy(host_stats, S.stats, sizeof S.stats);
    return TS_OK;
}

int ts_render_controls_r(const ts_voice *d_params, int B, int sr, double seconds, int R, double *d_ctl) {
    if (!d_params || !d_ctl) return fail(TS_ENULL, "NULL argument%s");
    if (R <= 0) return fail(TS_EINVAL, "R must be positive%s");
    return render_impl(const_cast<ts_voice *>(d_params), sample_spec{false, 0, 0}, B, sr, seconds, TS_F32, nullptr, nullptr, 4, d_ctl, R);
}
int ts_render_r(const ts_voice *d_params, int B, int sr, double seconds, int R, float *d_audio) {
    if (!d_params || !d_audio) return fail(TS_ENULL, "NULL argument%s");
    if (R == TS_R) return ts_render_fmt(d_params, B, sr, seconds, TS_F32, d_audio, nullptr);
    if (R != 1) return fail(TS_EINVAL, "the audio path is built for R = 100 and R = 1%s");
    if (S.corpus.open) return fail(TS_EINVAL, "close the corpus iterator first%s");
    S.cur = &S.lane[0];
    return render_impl(const_cast<ts_voice *>(d_params), sample_spec{false, 0, 0}, B, sr, seconds, TS_F32, d_audio, nullptr, 5, nullptr, 1);
}
int ts_render_controls(const ts_voice *d_params, int B, int sr, double seconds, double *d_ctl) {
    return ts_render_controls_r(d_params, B, sr, seconds, TS_R, d_ctl);
}

static int mmd_impl(const float *d_x, const float *d_y, int n, int d, double *d_out, int pairwise) {
    if (!d_x || !d_y || !d_out) return fail(TS_ENULL, "NULL argument%s");
    if (n <= 0 || d <= 0 || n > 65535) return fail(TS_EINVAL, "n must be in [1, 65535] and d positive%s");
    const size_t need = ts_mmd_partial_count(n, d);
    if (need > S.mmd_ws_count) {
        if (S.mmd_ws) {
            cudaStreamSynchronize(S.lane[0].stream);  // an earlier call may still use the old workspace
            cudaFree(S.mmd_ws);
        }
        S.mmd_ws = nullptr;
        S.mmd_ws_count = 0;
        if (cudaMalloc(&S.mmd_ws, need * sizeof(double)) != cudaSuccess) {
            cudaGetLastError();
            return fail(TS_ENOMEM, "MMD workspace allocation failed%s");
        }
        S.mmd_ws_count = need;
    }
    TS_CUDA(ts_launch_mmd(d_x, d_y, n, d, S.mmd_ws, d_out, pairwise, S.lane[0].stream));
    return TS_OK;
}
int ts_mmd_l1(const float *d_x, const float *d_y, int n, int d, double *d_out) { return mmd_impl(d_x, d_y, n, d, d_out, 0); }
int ts_mmd_l1_pairwise(const float *d_x, const float *d_y, int n, int d, double *d_out) { return mmd_impl(d_x, d_y, n, d, d_out, 1); }
int ts_mmd_l1_sorted(const float *d_x, const float *d_y, int n, int d, double *d_out) { return mmd_impl(d_x, d_y, n, d, d_out, 2); }

// ts_mmd_l1 for callers that cannot allocate: the scratch is a static device array of ts_mmd.cu (see there and tsynth.h).
// Touches none of the library's allocated state (S.mmd_ws stays as it is); no cudaMalloc / cudaFree on this path.
int ts_mmd_l1_static(const float *d_x, const float *d_y, int n, int d, double *d_out) {
    if (!d_x || !d_y || !d_out) return fail(TS_ENULL, "NULL argument%s");
    if (n <= 0 || d <= 0 || n > 65535) return fail(TS_EINVAL, "n must be in [1, 65535] and d positive%s");
    const size_t need = ts_mmd_partial_count(n, d), cap = ts_mmd_static_capacity();
    if (need > cap) {
        char detail[160];
        snprintf(detail, sizeof detail, "n = %d, d = %d needs %zu partial sums, the static scratch holds %zu (n <= 4032 and d <= 10922)",
                 n, d, need, cap);
        return fail(TS_EINVAL, "ts_mmd_l1_static: %s; use ts_mmd_l1, which allocates its workspace", detail);
    }
    TS_CUDA(ts_launch_mmd_static(d_x, d_y, n, d, d_out, S.lane[0].stream));
    return TS_OK;
}

int ts_debug_noise_u32(const uint32_t host_key[2], uint64_t n0, int count, uint32_t *d_out) {
    if (!host_key || !d_out) return fail(TS_ENULL, "NULL argument%s");
    if (count <= 0) return fail(TS_EINVAL, "count must be positive%s");
    TS_CUDA(ts_launch_noise_debug(host_key[0], host_key[1], n0, count, d_out, S.cur->stream));
    return TS_OK;
}
int ts_debug_controls(const ts_voice *d_params, int B, int sr, double seconds, double *d_ctl) {
    if (!d_params || !d_ctl) return fail(TS_ENULL, "NULL argument%s");
    return render_impl(const_cast<ts_voice *>(d_params), sample_spec{false, 0, 0}, B, sr, seconds, TS_F32, nullptr, nullptr, 3, d_ctl);
}
int ts_debug_phase(const ts_voice *d_params, int B, int sr, double seconds, int vco, double *d_phase) {
    if (!d_params || !d_phase) return fail(TS_ENULL, "NULL argument%s");
    if (vco != 1 && vco != 2) return fail(TS_EINVAL, "vco must be 1 or 2%s");
    return render_impl(const_cast<ts_voice *>(d_params), sample_spec{false, 0, 0}, B, sr, seconds, TS_F32, nullptr, nullptr, vco, d_phase);
}

}  // extern "C"
