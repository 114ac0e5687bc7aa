// ts_audio.cu -- the fused audio-rate kernel (S8..S14): upsample -> VCO phase accumulation -> sine and
// square/saw oscillators -> Philox white noise -> VCAs -> mixer -> one store per sample.
// P:L117 (audio-rate modules), P:L123 (module census, upsampling); BASELINE.json north_star (3), (4).
//
// Thread = one run of TS_RUN = 20 consecutive samples inside one control interval; CTA = 128 runs =
// one contiguous 2560-sample tile of one voice.  A run starts from its tick's table entry (phase from
// the control kernel's exact integer scan) and walks its samples serially:
//     phi += w;  w += w*e1            (fp64: increments are geometric inside an interval)
// so no thread ever waits for another.  Everything downstream of the reduced phase is fp32.
// The tile is staged in shared memory (conflict-free STS.128) and leaves the SM as ONE bulk
// asynchronous copy (cp.async.bulk, the TMA engine), i.e. fully coalesced 10 KB writes.
// Tiles past the voice's last audible sample are written as zeros without any arithmetic.
#include "ts_common.cuh"

namespace {

constexpr double MAGIC32 = 1572864.0;  // 1.5 * 2^20: ulp 2^-32 -> low word = signed Q0.32 of frac(phi)
constexpr double MAGIC33 = 786432.0;   // 1.5 * 2^19: ulp 2^-33 -> low word = signed Q0.32 of frac(2 phi)

__device__ __forceinline__ float ts_ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float ts_rcp(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ void ts_bulk_store(void *gdst, const void *ssrc, uint32_t bytes) {
    const uint32_t s = (uint32_t)__cvta_generic_to_shared(ssrc);
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(s), "r"(bytes)
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

// sin(th) for th in [-pi/2, pi/2], odd polynomial: relative accuracy ~1e-7 down to th -> 0, which
// the square/saw needs (its tanh has slope up to ~1e5 per cycle at the zero crossings, H4).
__device__ __forceinline__ float ts_sin_poly(float th) {
    const float t2 = th * th;
    float p = -2.5052108e-8f;                // -1/11!
    p = fmaf(p, t2, 2.7557319e-6f);          //  1/9!
    p = fmaf(p, t2, -1.9841270e-4f);         // -1/7!
    p = fmaf(p, t2, 8.3333333e-3f);          //  1/5!
    p = fmaf(p, t2, -1.6666667e-1f);         // -1/3!
    return fmaf(th * t2, p, th);
}

template <int MODE>
__global__ void __launch_bounds__(TS_AUDIO_THREADS)
ts_audio_kernel(const ts_tick *__restrict__ table, const ts_vhdr *__restrict__ hdr, int B, long long N, int K,
                float *__restrict__ audio, double *__restrict__ dbg_phase, int aligned) {
    __shared__ __align__(128) float4 stage[TS_TILE / 4];

    const int voice = blockIdx.x % B;  // time-major grid: the audible (expensive) tiles are dispatched first
    const long long tile = blockIdx.x / B;
    const long long n_tile0 = tile * TS_TILE;
    const int tid = threadIdx.x;
    const ts_vhdr hd = hdr[voice];
    const long long rem = N - n_tile0;
    const int count = (rem < TS_TILE) ? (int)rem : TS_TILE;  // samples of this tile inside the buffer
    float *row = audio + (size_t)voice * N + n_tile0;

    if (MODE == 0 && n_tile0 >= hd.n_act) {  // silent tile: exact zeros (S4 release over; pin P9)
        if (aligned) {
            float4 *r4 = reinterpret_cast<float4 *>(row);
            for (int i = tid; i < count / 4; i += TS_AUDIO_THREADS) r4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        } else {
            for (int i = tid; i < count; i += TS_AUDIO_THREADS) row[i] = 0.f;
        }
        return;
    }

    const long long r = tile * TS_AUDIO_THREADS + tid;  // run index inside the voice
    const long long n0 = r * TS_RUN;
    float4 *my = &stage[tid * (TS_RUN / 4)];

    if (n0 < hd.n_act || (MODE != 0 && n0 < N)) {
        const int j = (int)(r / TS_RUNS_PER_TICK);
        const int q = (int)(r - (long long)j * TS_RUNS_PER_TICK);
        const ts_tick *tk = table + (size_t)voice * K + j;
        const double2 *t2 = reinterpret_cast<const double2 *>(tk);
        const double2 v0 = __ldg(t2 + 0), v1 = __ldg(t2 + 1), v2 = __ldg(t2 + 2), v3 = __ldg(t2 + 3);
        const float4 A0 = __ldg(reinterpret_cast<const float4 *>(&tk[0].a1));
        const float4 A1 = __ldg(reinterpret_cast<const float4 *>(&tk[1].a1));

        double p1 = v0.x, w1 = v0.y, p2 = v2.x, w2 = v2.y;
        const double e1a = v1.x, e1b = v3.x;
        {   // hop to the q-th run of the interval: 20 samples per hop in closed form
            const double g1 = v1.y, g2 = v3.y;
            const double e20a = e1a * g1, e20b = e1b * g2;
            for (int i = 0; i < q; ++i) {
                p1 = fma(w1, g1, p1);
                w1 = fma(w1, e20a, w1);
                p2 = fma(w2, g2, p2);
                w2 = fma(w2, e20b, w2);
            }
        }
        // S8: linear upsampling of the three gain rows, as a running sum over the run
        const float mf = (float)(q * TS_RUN) * (1.0f / TS_R);
        const float da1 = (A1.x - A0.x) * (1.0f / TS_R), da2 = (A1.y - A0.y) * (1.0f / TS_R),
                    da3 = (A1.z - A0.z) * (1.0f / TS_R);
        float a1 = fmaf(A1.x - A0.x, mf, A0.x), a2 = fmaf(A1.y - A0.y, mf, A0.y), a3 = fmaf(A1.z - A0.z, mf, A0.z);
        const float shape = hd.shape, tanh_c = hd.tanh_c;
        const uint32_t blk0 = (uint32_t)(n0 >> 2);

#pragma unroll
        for (int g = 0; g < TS_RUN / 4; ++g) {
            uint32_t nz[4];
            if (MODE == 0) ts_philox4x32_10(blk0 + g, 0u, 0u, 1u, hd.nk0, hd.nk1, nz);  // S12
            float o[4];
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                if (MODE == 0) {
                    // ---- S10 sine VCO: frac(phi) as signed Q0.32 straight from the fp64 mantissa
                    const int x1 = __double2loint(p1 + MAGIC32);
                    const float y1 = __sinf((float)x1 * 1.4629180792671596e-9f);  // 2 pi 2^-32
                    // ---- S11 square/saw VCO: reduce to the nearest half cycle (H4)
                    const double t = p2 + MAGIC33;
                    const int lo = __double2loint(t), hi = __double2hiint(t);
                    const uint32_t sgn = (((uint32_t)hi << 31) ^ (uint32_t)lo) & 0x80000000u;
                    const float th = (float)lo * 7.314590396335798e-10f;  // 2 pi 2^-33, th in [-pi/2, pi/2)
                    const float sn = __uint_as_float(__float_as_uint(ts_sin_poly(th)) ^ sgn);
                    const float cs = __uint_as_float(__float_as_uint(__cosf(th)) ^ sgn);
                    const float ex = ts_ex2(tanh_c * sn);
                    const float th2 = fmaf(-2.0f, ts_rcp(1.0f + ex), 1.0f);  // tanh((pi/2) k sin)
                    const float y2 = th2 * fmaf(shape, cs, 1.0f);
                    // ---- S12 noise value, S13 VCAs, S14 mixer (gains already carry the mixer levels)
                    const float z = fmaf((float)(nz[s] >> 8), 1.0f / 8388608.0f, -1.0f);
                    o[s] = fmaf(a3, z, fmaf(a2, y2, a1 * y1));
                    a1 += da1; a2 += da2; a3 += da3;
                } else {
                    const long long n = n0 + g * 4 + s;
                    const double ph = (MODE == 1) ? p1 : p2;
                    if (n < N) dbg_phase[(size_t)voice * N + n] = ph - floor(ph);
                }
                // ---- S9: phase accumulation; increments are geometric inside the interval
                p1 += w1; w1 = fma(w1, e1a, w1);
                p2 += w2; w2 = fma(w2, e1b, w2);
            }
            if (MODE == 0) my[g] = make_float4(o[0], o[1], o[2], o[3]);
        }
    } else if (MODE == 0) {
#pragma unroll
        for (int g = 0; g < TS_RUN / 4; ++g) my[g] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    if (MODE != 0) return;

    if (aligned) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> async proxy
        __syncthreads();
        if (tid == 0) ts_bulk_store(row, stage, (uint32_t)count * 4u);
    } else {
        __syncthreads();
        const float *sf = reinterpret_cast<const float *>(stage);
        for (int i = tid; i < count; i += TS_AUDIO_THREADS) row[i] = sf[i];
    }
}

}  // namespace

cudaError_t ts_launch_audio(const ts_tick *table, const ts_vhdr *hdr, int B, int64_t N, int K, float *audio,
                            int mode, double *dbg_phase, cudaStream_t st) {
    const int64_t tiles = (N + TS_TILE - 1) / TS_TILE;
    const int64_t grid = tiles * B;
    if (grid > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int aligned = (N % 4 == 0) && ((reinterpret_cast<uintptr_t>(audio) & 15u) == 0);
    if (mode == 0)
        ts_audio_kernel<0><<<(unsigned)grid, TS_AUDIO_THREADS, 0, st>>>(table, hdr, B, N, K, audio, dbg_phase, aligned);
    else if (mode == 1)
        ts_audio_kernel<1><<<(unsigned)grid, TS_AUDIO_THREADS, 0, st>>>(table, hdr, B, N, K, audio, dbg_phase, 0);
    else
        ts_audio_kernel<2><<<(unsigned)grid, TS_AUDIO_THREADS, 0, st>>>(table, hdr, B, N, K, audio, dbg_phase, 0);
    return cudaGetLastError();
}
