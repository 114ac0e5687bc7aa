// ts_api.cu -- the C-ABI of include/tsynth.h: argument checks, the nebula, the workspace (control tables
// sized to stay L2-resident), voice chunking and kernel launches.  No arithmetic of the method lives here.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include "ts_common.cuh"

namespace {

// A lane = a workspace with the stream(s) that use it, so that two batches can be in flight at once.
// Lane 0 serves ts_render / ts_render_host on the caller's stream.  Lanes 1 and 2 serve ts_corpus_render: they
// share one HIGH-priority stream for the sampler and the (latency-bound) control kernel and one LOW-priority
// stream for the (issue-bound) audio kernel, so that the control stage of batch i+1 is dispatched into the SMs
// while the audio stage of batch i still runs and fills the issue slots it leaves idle.
struct ts_lane {
    cudaStream_t stream = nullptr;
    void *ws = nullptr;
    size_t ws_bytes = 0;
    unsigned int epoch = 0;  // look-back flag value of the latest control launch on this workspace
    unsigned long long *d_active = nullptr;
    unsigned long long *h_active = nullptr;  // pinned
    // lanes 1, 2 (ts_corpus_render): the audio kernel goes to its own low-priority stream
    cudaStream_t audio_stream = nullptr;
    cudaEvent_t ctl_done = nullptr, aud_done = nullptr;
    bool aud_pending = false;  // aud_done was recorded after the latest audio kernel that reads this workspace
};
constexpr int TS_LANES = 3;

struct ts_state {
    char err[512] = "";
    ts_range nebula[TS_NPARAM];
    bool nebula_init = false;
    bool nebula_dirty = true;  // device copy is stale
    bool math_uploaded = false;
    ts_lane lane[TS_LANES];
    ts_lane *cur = &lane[0];
    cudaEvent_t fork = nullptr;
    cudaStream_t hi = nullptr, lo = nullptr;  // ts_corpus_render's internal streams
    // host staging for ts_render_host
    void *stage = nullptr;
    size_t stage_bytes = 0;
    // timing / stats
    bool timing = false;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    float ms[2] = {0.f, 0.f};
    int64_t stats[3] = {0, 0, 0};
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

void ensure_nebula() {
    if (!S.nebula_init) {
        default_nebula(S.nebula);
        S.nebula_init = true;
        S.nebula_dirty = true;
    }
}

// The audio kernel reads frac(phase) out of the fp64 mantissa after adding 1.5*2^19, which needs the
// phase advance over one control interval to stay below 2^18 cycles (1.5*2^19 +- 2^18 keeps its exponent).
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
int tails_expected(double seconds) {
    const ts_range *n = S.nebula;
    auto hi = [&](int i) { return fmax(n[i].lo, n[i].hi); };
    const double t_end = hi(1) + fmax(fmax(hi(5), hi(10)), fmax(hi(15), hi(25)));
    return t_end < 0.8 * seconds;
}

int ensure_ws(size_t bytes) {
    if (bytes <= S.cur->ws_bytes) return TS_OK;
    if (S.cur->ws) cudaFree(S.cur->ws);
    S.cur->ws = nullptr;
    S.cur->ws_bytes = 0;
    if (cudaMalloc(&S.cur->ws, bytes) != cudaSuccess) {
        cudaGetLastError();
        return fail(TS_ENOMEM, "workspace allocation failed%s");
    }
    S.cur->ws_bytes = bytes;
    // look-back flags must never equal a future epoch: start from zeros and restart the epoch count
    if (cudaMemsetAsync(S.cur->ws, 0, bytes, S.cur->stream) != cudaSuccess) return cuda_fail(cudaGetLastError(), "cudaMemsetAsync");
    S.cur->epoch = 0;
    return TS_OK;
}

int chunk_voices(int B, int K) {
    size_t per = (size_t)K * sizeof(ts_tick);
    size_t c = TS_TABLE_BUDGET / per;
    if (c < 1) c = 1;
    if (c > (size_t)B) c = (size_t)B;
    return (int)c;
}
size_t ws_layout(int Bc, int K, size_t *off_hdr, size_t *off_agg = nullptr) {
    size_t table = ((size_t)Bc * K * sizeof(ts_tick) + 255) & ~(size_t)255;
    if (off_hdr) *off_hdr = table;
    size_t agg = table + (((size_t)Bc * sizeof(ts_vhdr) + 255) & ~(size_t)255);
    if (off_agg) *off_agg = agg;
    return agg + ((ts_control_agg_bytes(Bc, K) + 255) & ~(size_t)255);
}

int check_sizes(int B, int sr, double seconds, int64_t *N, int *K) {
    if (B <= 0 || sr <= 0 || !(seconds > 0.0)) return fail(TS_EINVAL, "B, sr and seconds must be positive%s");
    const double ns = (double)sr * seconds;
    if (!(ns < 2.0e9)) return fail(TS_EINVAL, "sr*seconds too large%s");
    *N = ts_num_samples(sr, seconds);
    if (*N <= 0) return fail(TS_EINVAL, "zero samples%s");
    *K = (int)ts_num_ticks(*N);
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
    if (!S.cur->d_active) {
        TS_CUDA(cudaMalloc(&S.cur->d_active, sizeof(unsigned long long)));
        TS_CUDA(cudaMallocHost(&S.cur->h_active, sizeof(unsigned long long)));
        *S.cur->h_active = 0;
    }
    return TS_OK;
}

// mode 0: audio (+ optional params_human); 1/2: debug phase of VCO 1/2; 3: debug controls only
int render_impl(const ts_voice *d_params, int B, int sr, double seconds, float *audio, float *params_human, int mode,
                double *dbg) {
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K);
    if (rc) return rc;
    rc = prepare_common(sr);
    if (rc) return rc;
    const int Bc = chunk_voices(B, K);
    size_t off_hdr, off_agg;
    rc = ensure_ws(ws_layout(Bc, K, &off_hdr, &off_agg));
    if (rc) return rc;
    ts_tick *table = reinterpret_cast<ts_tick *>(S.cur->ws);
    ts_vhdr *hdr = reinterpret_cast<ts_vhdr *>(static_cast<char *>(S.cur->ws) + off_hdr);
    void *agg = static_cast<char *>(S.cur->ws) + off_agg;

    if (S.timing && mode == 0)
        for (auto &e : S.ev)
            if (!e) TS_CUDA(cudaEventCreate(&e));
    S.ms[0] = S.ms[1] = 0.f;
    int64_t launches = 0, chunks = 0;
    const bool want_stats = S.timing;  // the active-sample count costs a memset and a copy per call
    if (want_stats) TS_CUDA(cudaMemsetAsync(S.cur->d_active, 0, sizeof(unsigned long long), S.cur->stream));
    if (mode == 3) TS_CUDA(cudaMemsetAsync(dbg, 0, (size_t)B * 5 * K * sizeof(double), S.cur->stream));

    for (int b0 = 0; b0 < B; b0 += Bc) {
        const int nb = (B - b0 < Bc) ? (B - b0) : Bc;
        const bool timed = S.timing && mode == 0;
        if (timed) TS_CUDA(cudaEventRecord(S.ev[0], S.cur->stream));
        if (S.cur->aud_pending) {  // the audio kernel still reading this workspace's table goes first
            TS_CUDA(cudaStreamWaitEvent(S.cur->stream, S.cur->aud_done, 0));
            S.cur->aud_pending = false;
        }
        if (++S.cur->epoch == 0) {  // wrapped after 2^32 launches: clear the flags and start over
            TS_CUDA(cudaMemsetAsync(agg, 0, ts_control_agg_bytes(Bc, K), S.cur->stream));
            S.cur->epoch = 1;
        }
        TS_CUDA(ts_launch_control(d_params + b0, nb, sr, N, K, table, hdr, agg, S.cur->epoch,
                                  params_human ? params_human + (size_t)b0 * TS_NPARAM : nullptr,
                                  mode == 3 ? dbg + (size_t)b0 * 5 * K : nullptr, want_stats ? S.cur->d_active : nullptr,
                                  (mode == 1 || mode == 2) ? 1 : 0, S.cur->stream));
        ++launches;
        if (timed) TS_CUDA(cudaEventRecord(S.ev[1], S.cur->stream));
        cudaStream_t ast = S.cur->stream;
        if (S.cur->audio_stream && mode == 0) {  // hand over to the audio stream
            ast = S.cur->audio_stream;
            TS_CUDA(cudaEventRecord(S.cur->ctl_done, S.cur->stream));
            TS_CUDA(cudaStreamWaitEvent(ast, S.cur->ctl_done, 0));
        }
        if (mode != 3) {
            TS_CUDA(ts_launch_audio(table, hdr, nb, N, K, audio ? audio + (size_t)b0 * N : nullptr, mode, tails_expected(seconds),
                                    (mode == 1 || mode == 2) ? dbg + (size_t)b0 * N : nullptr, ast));
            ++launches;
        }
        if (ast != S.cur->stream) {  // the next control launch on this workspace will wait for this audio kernel
            TS_CUDA(cudaEventRecord(S.cur->aud_done, ast));
            S.cur->aud_pending = true;
        }
        if (timed) {
            TS_CUDA(cudaEventRecord(S.ev[2], S.cur->stream));
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
        TS_CUDA(cudaMemcpyAsync(S.cur->h_active, S.cur->d_active, sizeof(unsigned long long), cudaMemcpyDeviceToHost,
                                S.cur->stream));
    S.stats[0] = launches;
    S.stats[1] = chunks;
    return TS_OK;
}

}  // namespace

extern "C" {

int ts_corpus_is_test(uint64_t g) { return (g / 1024u) % 10u == 9u; }

int64_t ts_num_samples(int sr, double seconds) { return (int64_t)llround((double)sr * seconds); }
int64_t ts_num_ticks(int64_t N) { return (N + TS_R - 1) / TS_R + 1; }

int ts_sample_params(uint64_t seed, uint64_t batch_index, int B, ts_voice *d_params) {
    if (!d_params) return fail(TS_ENULL, "d_params is NULL%s");
    if (B <= 0) return fail(TS_EINVAL, "B must be positive%s");
    TS_CUDA(ts_launch_sample(seed, batch_index * (uint64_t)B, B, d_params, S.cur->stream));
    return TS_OK;
}

int ts_render(const ts_voice *d_params, int B, int sr, double seconds, ts_out out) {
    if (!d_params) return fail(TS_ENULL, "d_params is NULL%s");
    if (!out.audio) return fail(TS_ENULL, "out.audio is NULL%s");
    return render_impl(d_params, B, sr, seconds, out.audio, out.params_human, 0, nullptr);
}

int ts_render_host(uint64_t seed, uint64_t batch_index, int B, int sr, double seconds, float *host_audio,
                   ts_voice *host_params) {
    if (!host_audio) return fail(TS_ENULL, "host_audio is NULL%s");
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K);
    if (rc) return rc;
    const size_t pbytes = ((size_t)B * sizeof(ts_voice) + 255) & ~(size_t)255;
    const size_t abytes = (size_t)B * N * sizeof(float);
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
    float *d_audio = reinterpret_cast<float *>(static_cast<char *>(S.stage) + pbytes);
    rc = ts_sample_params(seed, batch_index, B, d_params);
    if (rc) return rc;
    rc = render_impl(d_params, B, sr, seconds, d_audio, nullptr, 0, nullptr);
    if (rc) return rc;
    TS_CUDA(cudaMemcpyAsync(host_audio, d_audio, abytes, cudaMemcpyDeviceToHost, S.cur->stream));
    if (host_params)
        TS_CUDA(cudaMemcpyAsync(host_params, d_params, (size_t)B * sizeof(ts_voice), cudaMemcpyDeviceToHost, S.cur->stream));
    TS_CUDA(cudaStreamSynchronize(S.cur->stream));
    return TS_OK;
}

int ts_corpus_render(uint64_t seed, uint64_t first_batch, int n_batches, int B, int sr, double seconds,
                     ts_voice *d_params_ring, float *d_audio_ring, int n_ring) {
    if (!d_params_ring || !d_audio_ring) return fail(TS_ENULL, "NULL ring%s");
    if (n_batches <= 0 || n_ring <= 0) return fail(TS_EINVAL, "n_batches and n_ring must be positive%s");
    int64_t N;
    int K;
    int rc = check_sizes(B, sr, seconds, &N, &K);
    if (rc) return rc;
    S.cur = &S.lane[0];
    rc = prepare_common(sr);  // nebula / tables go up on the caller's stream, before the fork
    if (rc) return rc;
    if (!S.fork) {
        int lo_p = 0, hi_p = 0;
        TS_CUDA(cudaDeviceGetStreamPriorityRange(&lo_p, &hi_p));  // numerically lower = higher priority
        TS_CUDA(cudaStreamCreateWithPriority(&S.hi, cudaStreamNonBlocking, hi_p));
        TS_CUDA(cudaStreamCreateWithPriority(&S.lo, cudaStreamNonBlocking, lo_p));
        for (int l = 1; l < TS_LANES; ++l) {
            S.lane[l].stream = S.hi;
            S.lane[l].audio_stream = S.lo;
            TS_CUDA(cudaEventCreateWithFlags(&S.lane[l].ctl_done, cudaEventDisableTiming));
            TS_CUDA(cudaEventCreateWithFlags(&S.lane[l].aud_done, cudaEventDisableTiming));
        }
        TS_CUDA(cudaEventCreateWithFlags(&S.fork, cudaEventDisableTiming));
    }
    // fork: both internal streams start after everything already queued on the caller's stream
    TS_CUDA(cudaEventRecord(S.fork, S.lane[0].stream));
    TS_CUDA(cudaStreamWaitEvent(S.hi, S.fork, 0));
    TS_CUDA(cudaStreamWaitEvent(S.lo, S.fork, 0));
    const bool timing = S.timing;
    S.timing = false;  // per-kernel events would serialise the streams
    // Ring hazards: records are written by the sampler and read by the control kernel, both on `hi` in batch order;
    // audio slots are written by the audio kernels, all on `lo` in batch order.  Nothing else to order.
    for (int i = 0; i < n_batches && rc == TS_OK; ++i) {
        ts_lane &L = S.lane[1 + (i & 1)];
        const size_t slot = (size_t)(i % n_ring);
        ts_voice *p = d_params_ring + slot * (size_t)B;
        float *a = d_audio_ring + slot * (size_t)B * (size_t)N;
        cudaError_t e = ts_launch_sample(seed, (first_batch + (uint64_t)i) * (uint64_t)B, B, p, L.stream);
        if (e != cudaSuccess) { rc = cuda_fail(e, "ts_launch_sample"); break; }
        S.cur = &L;
        rc = render_impl(p, B, sr, seconds, a, nullptr, 0, nullptr);
    }
    S.cur = &S.lane[0];
    S.timing = timing;
    // join: the caller's stream continues after both internal streams
    TS_CUDA(cudaEventRecord(S.lane[1].ctl_done, S.hi));
    TS_CUDA(cudaStreamWaitEvent(S.lane[0].stream, S.lane[1].ctl_done, 0));
    TS_CUDA(cudaEventRecord(S.lane[2].ctl_done, S.lo));
    TS_CUDA(cudaStreamWaitEvent(S.lane[0].stream, S.lane[2].ctl_done, 0));
    S.stats[0] *= n_batches;  // kernels launched by this call (3 per batch and voice chunk: sampler counted below)
    S.stats[0] += n_batches;
    return rc;
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
    if (!host_in78) {
        default_nebula(S.nebula);
    } else {
        for (int i = 0; i < TS_NPARAM; ++i) {
            const ts_range &r = host_in78[i];
            if (!(r.curve > 0.0) || !isfinite(r.lo) || !isfinite(r.hi) || !isfinite(r.curve))
                return fail(TS_EINVAL, "nebula entries must be finite with curve > 0%s");
        }
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
    return ws_layout(chunk_voices(B, K), K, nullptr);
}

const char *ts_last_error(void) { return S.err; }

int ts_sync(void) {
    TS_CUDA(cudaStreamSynchronize(S.lane[0].stream));
    if (S.lane[0].h_active) S.stats[2] = (int64_t)*S.lane[0].h_active;
    return TS_OK;
}

void ts_shutdown(void) {
    for (int l = 0; l < TS_LANES; ++l) {
        ts_lane &L = S.lane[l];
        if (L.ws) cudaFree(L.ws);
        if (L.d_active) cudaFree(L.d_active);
        if (L.h_active) cudaFreeHost(L.h_active);
        if (L.ctl_done) cudaEventDestroy(L.ctl_done);
        if (L.aud_done) cudaEventDestroy(L.aud_done);
        const cudaStream_t keep = (l == 0) ? L.stream : nullptr;
        L = ts_lane();
        L.stream = keep;
    }
    if (S.fork) { cudaEventDestroy(S.fork); S.fork = nullptr; }
    if (S.hi) { cudaStreamDestroy(S.hi); S.hi = nullptr; }
    if (S.lo) { cudaStreamDestroy(S.lo); S.lo = nullptr; }
    if (S.stage) cudaFree(S.stage);
    for (auto &e : S.ev)
        if (e) { cudaEventDestroy(e); e = nullptr; }
    S.stage = nullptr;
    S.stage_bytes = 0;
    S.cur = &S.lane[0];
    S.nebula_dirty = true;
    S.math_uploaded = false;
}

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
    const int Bc = chunk_voices(B, K);
    size_t off_hdr, off_agg;
    rc = ensure_ws(ws_layout(Bc, K, &off_hdr, &off_agg));
    if (rc) return rc;
    ts_tick *table = reinterpret_cast<ts_tick *>(S.cur->ws);
    ts_vhdr *hdr = reinterpret_cast<ts_vhdr *>(static_cast<char *>(S.cur->ws) + off_hdr);
    void *agg = static_cast<char *>(S.cur->ws) + off_agg;
    for (auto &e : S.ev)
        if (!e) TS_CUDA(cudaEventCreate(&e));
    cudaStream_t st = S.cur->stream;
    float a = 0.f, b = 0.f;
    for (int b0 = 0; b0 < B; b0 += Bc) {  // voice chunk by voice chunk, as ts_render launches them
        const int nb = (B - b0 < Bc) ? (B - b0) : Bc;
        TS_CUDA(cudaEventRecord(S.ev[0], st));
        for (int r = 0; r < reps; ++r) {
            if (++S.cur->epoch == 0) {
                TS_CUDA(cudaMemsetAsync(agg, 0, ts_control_agg_bytes(Bc, K), st));
                S.cur->epoch = 1;
            }
            TS_CUDA(ts_launch_control(d_params + b0, nb, sr, N, K, table, hdr, agg, S.cur->epoch, nullptr, nullptr, nullptr, 0,
                                      st));
        }
        TS_CUDA(cudaEventRecord(S.ev[1], st));
        for (int r = 0; r < reps; ++r)
            TS_CUDA(ts_launch_audio(table, hdr, nb, N, K,
                                    d_audio_ring + (size_t)(r % n_ring) * (size_t)B * (size_t)N + (size_t)b0 * (size_t)N, 0,
                                    tails_expected(seconds), nullptr, st));
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

int ts_debug_noise_u32(const uint32_t host_key[2], uint64_t n0, int count, uint32_t *d_out) {
    if (!host_key || !d_out) return fail(TS_ENULL, "NULL argument%s");
    if (count <= 0) return fail(TS_EINVAL, "count must be positive%s");
    TS_CUDA(ts_launch_noise_debug(host_key[0], host_key[1], n0, count, d_out, S.cur->stream));
    return TS_OK;
}
int ts_debug_controls(const ts_voice *d_params, int B, int sr, double seconds, double *d_ctl) {
    if (!d_params || !d_ctl) return fail(TS_ENULL, "NULL argument%s");
    return render_impl(d_params, B, sr, seconds, nullptr, nullptr, 3, d_ctl);
}
int ts_render_controls(const ts_voice *d_params, int B, int sr, double seconds, double *d_ctl) {
    return ts_debug_controls(d_params, B, sr, seconds, d_ctl);
}
int ts_debug_phase(const ts_voice *d_params, int B, int sr, double seconds, int vco, double *d_phase) {
    if (!d_params || !d_phase) return fail(TS_ENULL, "NULL argument%s");
    if (vco != 1 && vco != 2) return fail(TS_EINVAL, "vco must be 1 or 2%s");
    return render_impl(d_params, B, sr, seconds, nullptr, nullptr, vco, d_phase);
}

}  // extern "C"
