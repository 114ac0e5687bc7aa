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
// Tiles past the voice's last audible sample are written as zeros without any arithmetic, by the voice's audible CTAs.
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

// The output is written once and not read again by this path: its lines are marked evict-first in L2, so that 90 MB of
// streaming stores per launch do not push the control table (read by every run, written by the control kernel just
// before) and the other lanes' working sets out of the 126 MB L2.  Measured on C2: audio kernel 24.6 -> 22.6 us, the
// same as with the silent tails not written at all.
__device__ __forceinline__ unsigned long long ts_policy_evict_first() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void ts_bulk_issue(void *gdst, uint32_t ssrc, uint32_t bytes) {  // TMA engine (UBLKCP)
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(gdst), "r"(ssrc), "r"(bytes),
                 "l"(ts_policy_evict_first())
                 : "memory");
}
__device__ __forceinline__ void ts_bulk_store(void *gdst, const void *ssrc, uint32_t bytes) {
    ts_bulk_issue(gdst, (uint32_t)__cvta_generic_to_shared(ssrc), bytes);
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

// ---- packed fp32x2 arithmetic (Blackwell FFMA2 / FMUL2 / FADD2): one issue slot for two samples -----
typedef unsigned long long ts_f2;
__device__ __forceinline__ ts_f2 ts_pack(float lo, float hi) {
    ts_f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void ts_unpack(ts_f2 v, float &lo, float &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ ts_f2 ts_fma2(ts_f2 a, ts_f2 b, ts_f2 c) {
    ts_f2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ ts_f2 ts_mul2(ts_f2 a, ts_f2 b) {
    ts_f2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ ts_f2 ts_add2(ts_f2 a, ts_f2 b) {
    ts_f2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ ts_f2 ts_dup(float c) { return ts_pack(c, c); }
// two fp32 samples -> one 32-bit word of two fp16 / bf16 samples (round to nearest even), first sample in the low half
template <int FMT> __device__ __forceinline__ uint32_t ts_cvt16(ts_f2 v) {
    float lo, hi;
    ts_unpack(v, lo, hi);
    uint32_t d;
    if (FMT == TS_F16) asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    else asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    return d;
}

// sin(th) for th in [-pi/2, pi/2] as th + th^3 q(th^2), q minimax of degree 3 (fit of (sin x / x - 1) / x^2 with
// relative weighting): relative accuracy 1.2e-7 in fp32 down to th -> 0, which the square/saw needs (its tanh
// has slope up to ~1e5 per cycle at the zero crossings, H4).
constexpr float SIN_C3 = -0.16666659712791443f, SIN_C5 = 0.008333087898790836f, SIN_C7 = -0.00019811101083178073f,
                SIN_C9 = 2.6089039693033556e-06f;
// The 20 samples of one run (S9..S14) from its start state, into the thread's slice of the staging tile.
// FASTSIN: the square/saw's sine through MUFU.SIN on the whole cycle instead of the relative-accuracy polynomial on the
// nearest half cycle.  The sine is multiplied by (pi/2) k before the tanh (S11), so its ABSOLUTE error at the zero
// crossings decides: near theta = +-pi the fp32 angle carries the rounding of the int -> float conversion, of the scaling
// and of sin.approx's own multiplication by 1/(2 pi) (together <= 3.8e-7 rad) and MUFU.SIN adds 2^-21.4 (3.6e-7):
// 7.4e-7.  Taken only for voices whose steepness k <= 512 (note frequency above 18.6 Hz: 89 % of the voices under the
// default nebula): the error it adds to a sample is then below (pi/2) 512 * 7.4e-7 * 1.125 = 6.7e-4, a third of the 2e-3
// bar, and only within ~1/k of a cycle around the zero crossings (rel-RMS contribution < 3e-5) (H4; the flag is set by
// the setup kernel).
template <int FMT, int FASTSIN>
__device__ __forceinline__ void ts_render_run(double P1, double w1, const double e1a, double P2, double w2, const double e1b,
                                              float a1, float a2, float a3, const float da1, const float da2, const float da3,
                                              const uint32_t blk0, const uint32_t nk0, const uint32_t nk1, const float shape,
                                              const float tanh_c, const uint32_t one_bits, float4 *my, uint2 *my16) {
        const ts_f2 SHAPE = ts_dup(shape), TANH_C = ts_dup(tanh_c), ONE = ts_dup(1.0f);
        ts_f2 G1 = ts_pack(a1, a1 + da1), G2 = ts_pack(a2, a2 + da2), G3 = ts_pack(a3, a3 + da3);
        const ts_f2 DG1 = ts_dup(2.0f * da1), DG2 = ts_dup(2.0f * da2), DG3 = ts_dup(2.0f * da3);
        ulonglong2 *my2 = reinterpret_cast<ulonglong2 *>(my);
        // S9 two samples at a time: the increments are geometric (w_{n+1} = rho w_n, rho = 1 + e1), so from (P_n, w_n)
        //     P_{n+1} = P_n + w_n,   P_{n+2} = P_n + w_n (1 + rho),   w_{n+2} = w_n rho^2 = w_n + w_n (2 e1 + e1^2)
        // three fp64 instructions per pair and oscillator instead of four
        const double c2a = 2.0 + e1a, c2b = 2.0 + e1b;
        const double e2a = fma(e1a, e1a, e1a + e1a), e2b = fma(e1b, e1b, e1b + e1b);
#pragma unroll
        for (int g = 0; g < TS_RUN / 4; ++g) {
            uint32_t nz[4];
            ts_philox4x32_10(blk0 + g, 0u, 0u, 1u, nk0, nk1, nz);  // S12
            ts_f2 O[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                // ---- S9: phase accumulation for two consecutive samples (fp64, geometric increments)
                const double P1b = P1 + w1, P2b = P2 + w2;
                const int xa = __double2loint(P1), xb = __double2loint(P1b);
                const int la = __double2loint(P2), lb = __double2loint(P2b);
                const int ha = __double2hiint(P2), hb = __double2hiint(P2b);
                P1 = fma(w1, c2a, P1); w1 = fma(w1, e2a, w1);
                P2 = fma(w2, c2b, P2); w2 = fma(w2, e2b, w2);
                // ---- S10 sine VCO: frac(phi) is the signed Q0.32 in the low word
                float r1a, r1b;
                ts_unpack(ts_mul2(ts_pack((float)xa, (float)xb), ts_dup(1.4629180792671596e-9f)), r1a, r1b);  // 2 pi 2^-32
                const ts_f2 Y1 = ts_pack(__sinf(r1a), __sinf(r1b));
                // ---- S11 square/saw VCO
                float ea, eb, da, db;
                float tha, thb;
                ts_f2 SN, SC;  // sin(theta) (up to the sign sigma), sigma + s cos(theta) (up to sigma)
                if (FASTSIN) {
                    // gentle voices (k <= TS_FASTSIN_K): the accumulator is biased like VCO 1's, its low word is the signed
                    // Q0.32 of the whole cycle, and MUFU.SIN / MUFU.COS take theta in [-pi, pi) as it is: no half-cycle
                    // parity, y2 = tanh(c sin theta) (1 + s cos theta) literally
                    ts_unpack(ts_mul2(ts_pack((float)la, (float)lb), ts_dup(1.4629180792671596e-9f)), tha, thb);  // 2 pi 2^-32
                    SN = ts_pack(__sinf(tha), __sinf(thb));
                    SC = ts_fma2(SHAPE, ts_pack(__cosf(tha), __cosf(thb)), ONE);
                } else {
                    // steep voices: low word = signed Q0.32 of the nearest HALF cycle (H4), so that theta -> 0 at BOTH zero
                    // crossings of the sine and the polynomial's relative accuracy holds there; the parity of that half
                    // cycle (bit 0 of the high word, +1 if the low word is negative) is the sign sigma, folded in as
                    // y2 = sigma tanh (1 + s sigma cos) = tanh (sigma + s cos)
                    const uint32_t sa = (((uint32_t)la + ((uint32_t)ha << 31)) & 0x80000000u) | one_bits;
                    const uint32_t sb = (((uint32_t)lb + ((uint32_t)hb << 31)) & 0x80000000u) | one_bits;
                    const ts_f2 SIG = ts_pack(__uint_as_float(sa), __uint_as_float(sb));
                    const ts_f2 TH = ts_mul2(ts_pack((float)la, (float)lb), ts_dup(7.314590396335798e-10f));  // 2 pi 2^-33
                    ts_unpack(TH, tha, thb);
                    const ts_f2 T2 = ts_mul2(TH, TH);
                    ts_f2 Q = ts_fma2(T2, ts_dup(SIN_C9), ts_dup(SIN_C7));
                    Q = ts_fma2(Q, T2, ts_dup(SIN_C5));
                    Q = ts_fma2(Q, T2, ts_dup(SIN_C3));
                    SN = ts_fma2(ts_mul2(TH, T2), Q, TH);
                    SC = ts_fma2(SHAPE, ts_pack(__cosf(tha), __cosf(thb)), SIG);
                }
                ts_unpack(ts_mul2(SN, TANH_C), ea, eb);
                ts_unpack(ts_add2(ts_pack(ts_ex2(ea), ts_ex2(eb)), ONE), da, db);
                // tanh((pi/2) k sin) = 1 - 2 / (1 + 2^(c sin))
                const ts_f2 TNH = ts_fma2(ts_pack(ts_rcp(da), ts_rcp(db)), ts_dup(-2.0f), ONE);
                const ts_f2 Y2 = ts_mul2(TNH, SC);
                // ---- S12 noise value (RZ conversion keeps the top 24 bits of x when x >= 2^31 and a few more
                // below: within 2^-24 of (x >> 8) 2^-23 - 1), S13 VCAs, S14 mixer (gains carry the mixer levels)
                const ts_f2 Z = ts_fma2(ts_pack(__uint2float_rz(nz[2 * h]), __uint2float_rz(nz[2 * h + 1])),
                                        ts_dup(4.656612873077393e-10f), ts_dup(-1.0f));
                O[h] = ts_fma2(G3, Z, ts_fma2(G2, Y2, ts_mul2(G1, Y1)));
                G1 = ts_add2(G1, DG1); G2 = ts_add2(G2, DG2); G3 = ts_add2(G3, DG3);
            }
            if (FMT == TS_F32) my2[g] = make_ulonglong2(O[0], O[1]);
            else my16[g] = make_uint2(ts_cvt16<FMT>(O[0]), ts_cvt16<FMT>(O[1]));
        }
}

// TAIL = 1: the silent tails are written by the audible CTAs (below); TAIL = 0: every silent tile is written by a CTA of
// its own (better when few tiles are silent: no zero buffer, more L1 left for the control table).
// FMT: output sample format (TS_F32 / TS_F16 / TS_BF16): the finished fp32 sample is rounded once, two samples per
// cvt.rn.{f16x2,bf16x2}.f32, on its way into the staging tile.
// TPC: consecutive tiles of one voice rendered by one CTA, one after the other (large launches: halves the CTA turnover,
// which costs ~14 % of an SM's time at one tile per CTA; small launches keep TPC = 1 so that the last wave stays short).
#ifndef TS_AUDIO_MINB
#define TS_AUDIO_MINB 10  // 48 registers: ten CTAs per SM (9 at 52 registers measured 2 % slower on C3, 11 CTAs with spills slower)
#endif
template <int MODE, int TAIL, int FMT, int TPC>
__global__ void __launch_bounds__(TS_AUDIO_THREADS, TS_AUDIO_MINB)
ts_audio_kernel(const ts_tick *__restrict__ table, const ts_vhdr *__restrict__ hdr, int B, int N, int K,
                void *__restrict__ audio_, double *__restrict__ dbg_phase, int aligned, uint32_t one_bits, int swap) {
    __shared__ __align__(128) float4 stage[TS_TILE / 4];
    __shared__ __align__(128) float4 zero[(MODE == 0 && TAIL) ? TS_TILE / 4 : 4];  // source of the tail's zero-fill bulk copies

    constexpr int ES = (FMT == TS_F32) ? 4 : 2;  // bytes per output sample
    char *audio = static_cast<char *>(audio_);
    // 2-D grid, no integer division: x = voice, y = tile (x runs fastest: time-major dispatch, the audible tiles of all
    // voices go first); swapped when a voice has more than 65535 tiles
    const int voice = swap ? blockIdx.y : blockIdx.x;
    // N < 2^31 (ts_api.cu check_sizes): sample, run and tile indices are 32-bit, only byte offsets are 64-bit
    const int tile_first = (int)(swap ? blockIdx.x : blockIdx.y) * TPC;
    const int tid = threadIdx.x;
    const ts_vhdr hd = hdr[voice];
    // TAIL = 1: a CTA whose first tile is past the voice's last audible sample has nothing to do (its tiles are written
    // by the voice's audible CTAs); it leaves before any other arithmetic.  Tile 0 always stays (it owns the tail of a
    // voice with no audible sample).
    if (MODE == 0 && TAIL && tile_first > 0 && tile_first * TS_TILE >= hd.n_act) return;
    const int T = (N + TS_TILE - 1) / TS_TILE;
    bool zeroed = false;  // the zero buffer is filled once per CTA
#pragma unroll 1
    for (int tt = 0; tt < TPC; ++tt) {
    const int tile = tile_first + tt;
    if (tile >= T) return;
    if (TPC > 1 && tt > 0) __syncthreads();  // the previous tile's bulk copy has read the staging tile (thread 0 waited)
    const int n_tile0 = tile * TS_TILE;
    const int rem = N - n_tile0;
    const int count = (rem < TS_TILE) ? rem : TS_TILE;  // samples of this tile inside the buffer
    char *row = audio + ((size_t)voice * (size_t)N + (size_t)n_tile0) * ES;

    if (MODE == 0 && !TAIL && n_tile0 >= hd.n_act) {  // silent tile: exact zeros (S4 release over; pin P9)
        if (aligned) {
            float4 *r4 = reinterpret_cast<float4 *>(row);
            for (int i = tid; i < count * ES / 16; i += TS_AUDIO_THREADS) __stcs(&r4[i], make_float4(0.f, 0.f, 0.f, 0.f));  // streaming
        } else if (FMT == TS_F32) {
            for (int i = tid; i < count; i += TS_AUDIO_THREADS) reinterpret_cast<float *>(row)[i] = 0.f;
        } else {
            for (int i = tid; i < count; i += TS_AUDIO_THREADS) reinterpret_cast<unsigned short *>(row)[i] = 0;
        }
        continue;
    }
    if (MODE == 0 && TAIL) {
        // Samples [n_act, N) are exactly 0 (S4 release over; pin P9).  The silent tiles of a voice are not rendered by
        // CTAs of their own: audible tile t of a voice with A audible tiles writes the silent tiles A + t, A + t + A, ...
        // as asynchronous bulk copies of a zero buffer (TMA engine), issued BEFORE its arithmetic, so that the stores
        // of the tails overlap the issue-bound arithmetic of the audible part instead of following it.
        int A = (hd.n_act + TS_TILE - 1) / TS_TILE;
        if (A < 1) A = 1;  // a voice with no audible sample: tile 0 renders zeros and owns the whole tail
        if (tile >= A) return;  // and so are all later tiles of this voice
        char *vrow = audio + (size_t)voice * (size_t)N * ES;
        if (A + tile >= T) {
            // no silent tile falls to this CTA
        } else if (aligned) {
            if (!zeroed) {
#pragma unroll
                for (int g = 0; g < TS_RUN / 4; ++g) zero[tid * (TS_RUN / 4) + g] = make_float4(0.f, 0.f, 0.f, 0.f);
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> async proxy
                __syncthreads();
                zeroed = true;
            }
            if ((tid & 31) == 0) {  // lane 0 of each warp issues every fourth copy
                const uint32_t zs = (uint32_t)__cvta_generic_to_shared(zero);
                for (int tz = A + tile + (tid >> 5) * A; tz < T; tz += (TS_AUDIO_THREADS / 32) * A) {
                    const int rz = N - tz * TS_TILE;
                    ts_bulk_issue(vrow + (size_t)tz * (TS_TILE * ES), zs, ((rz < TS_TILE) ? (uint32_t)rz : (uint32_t)TS_TILE) * ES);
                }
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
        } else {
            for (int tz = A + tile; tz < T; tz += A) {
                const int rz = N - tz * TS_TILE;
                const int cz = (rz < TS_TILE) ? rz : TS_TILE;
                if (FMT == TS_F32)
                    for (int i = tid; i < cz; i += TS_AUDIO_THREADS) reinterpret_cast<float *>(vrow)[(size_t)tz * TS_TILE + i] = 0.f;
                else
                    for (int i = tid; i < cz; i += TS_AUDIO_THREADS) reinterpret_cast<unsigned short *>(vrow)[(size_t)tz * TS_TILE + i] = 0;
            }
        }
    }

    const int r = tile * TS_AUDIO_THREADS + tid;  // run index inside the voice
    const int n0 = r * TS_RUN;
    // this thread's 20 samples inside the staging tile: 80 bytes (fp32) or 40 bytes (16-bit formats), conflict-free
    float4 *my = &stage[tid * (TS_RUN / 4)];
    uint2 *my16 = reinterpret_cast<uint2 *>(reinterpret_cast<char *>(stage) + tid * (TS_RUN * 2));

    if (n0 < hd.n_act || (MODE != 0 && n0 < N)) {
        const int j = r / TS_RUNS_PER_TICK;
        const int q = r - j * TS_RUNS_PER_TICK;
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
#pragma unroll 1
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
        const uint32_t blk0 = (uint32_t)(n0 >> 2);
        // Biased accumulators: P = MAGIC + phi keeps frac(phi) in the low mantissa word at every step (the add
        // rounds to 2^-32 / 2^-33 of a cycle: <= 20 * 2^-33 = 2.3e-9 cycles over a run, budget 1e-8, H4).
        double P1 = p1 + MAGIC32, P2 = p2 + MAGIC33;

        if (MODE == 0) {
            if (hd.pad[0])  // CTA-uniform: the voice's square/saw is gentle enough for MUFU.SIN on the whole cycle
                ts_render_run<FMT, 1>(P1, w1, e1a, p2 + MAGIC32, w2, e1b, a1, a2, a3, da1, da2, da3, blk0, hd.nk0, hd.nk1, hd.shape, hd.tanh_c,
                                      one_bits, my, my16);
            else
                ts_render_run<FMT, 0>(P1, w1, e1a, P2, w2, e1b, a1, a2, a3, da1, da2, da3, blk0, hd.nk0, hd.nk1, hd.shape, hd.tanh_c,
                                      one_bits, my, my16);
        } else {
            for (int i = 0; i < TS_RUN; ++i) {
                const int n = n0 + i;
                const double ph = (MODE == 1) ? (P1 - MAGIC32) : (P2 - MAGIC33);
                if (n < N) dbg_phase[(size_t)voice * (size_t)N + n] = ph - floor(ph);
                P1 += w1; w1 = fma(w1, e1a, w1);
                P2 += w2; w2 = fma(w2, e1b, w2);
            }
        }
    } else if (MODE == 0) {
#pragma unroll
        for (int g = 0; g < TS_RUN / 4; ++g) {
            if (FMT == TS_F32) my[g] = make_float4(0.f, 0.f, 0.f, 0.f);
            else my16[g] = make_uint2(0u, 0u);
        }
    }
    if (MODE != 0) continue;

    if (aligned) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> async proxy
        __syncthreads();
        if (tid == 0) ts_bulk_store(row, stage, (uint32_t)count * ES);
        else if (TAIL && (tid & 31) == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");  // zero buffer still being read
    } else {
        __syncthreads();
        if (FMT == TS_F32) {
            const float *sf = reinterpret_cast<const float *>(stage);
            for (int i = tid; i < count; i += TS_AUDIO_THREADS) reinterpret_cast<float *>(row)[i] = sf[i];
        } else {
            const unsigned short *sh = reinterpret_cast<const unsigned short *>(stage);
            for (int i = tid; i < count; i += TS_AUDIO_THREADS) reinterpret_cast<unsigned short *>(row)[i] = sh[i];
        }
    }
    }  // tiles of this CTA
}

// ---- audio-rate-control mode (R = 1): every sample is a control tick, so there is no upsampling
// (pin P7) and no recurrence: a sample's phases and gains are its own table entry.  One thread renders the four samples of
// one Philox block.  A mode for studying the two-rate design (D1), not the hot path: plain fp32 arithmetic, the
// relative-accuracy polynomial for the square/saw sine, 128-bit stores when the row is aligned.
__global__ void __launch_bounds__(128)
ts_audio_r1_kernel(const ts_tick *__restrict__ table, const ts_vhdr *__restrict__ hdr, int B, int N, int K,
                   float *__restrict__ audio, int aligned, uint32_t one_bits) {
    const int voice = blockIdx.y;
    const int n0 = (blockIdx.x * 128 + threadIdx.x) * 4;
    if (n0 >= N) return;
    const ts_vhdr hd = hdr[voice];
    float o[4] = {0.f, 0.f, 0.f, 0.f};
    if (n0 < hd.n_act) {
        uint32_t nz[4];
        ts_philox4x32_10((uint32_t)(n0 >> 2), 0u, 0u, 1u, hd.nk0, hd.nk1, nz);  // S12
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int n = n0 + i;
            if (n >= hd.n_act || n >= N) continue;
            const ts_tick *tk = table + (size_t)voice * K + n;
            const double P1 = __ldg(&tk->phi1) + MAGIC32, P2 = __ldg(&tk->phi2) + MAGIC33;
            const float4 g = __ldg(reinterpret_cast<const float4 *>(&tk->a1));
            const int xa = __double2loint(P1), la = __double2loint(P2), ha = __double2hiint(P2);
            const float y1 = __sinf((float)xa * 1.4629180792671596e-9f);                                    // S10
            const uint32_t sg = (((uint32_t)la + ((uint32_t)ha << 31)) & 0x80000000u) | one_bits;       // S11 (H4)
            const float th = (float)la * 7.314590396335798e-10f, t2 = th * th;
            float q = fmaf(t2, SIN_C9, SIN_C7);
            q = fmaf(q, t2, SIN_C5);
            q = fmaf(q, t2, SIN_C3);
            const float sn = fmaf(th * t2, q, th);
            const float tnh = fmaf(ts_rcp(ts_ex2(sn * hd.tanh_c) + 1.0f), -2.0f, 1.0f);
            const float y2 = tnh * fmaf(hd.shape, __cosf(th), __uint_as_float(sg));
            const float z = fmaf(__uint2float_rz(nz[i]), 4.656612873077393e-10f, -1.0f);                  // S12, D24
            o[i] = fmaf(g.z, z, fmaf(g.y, y2, g.x * y1));                                                  // S13, S14
        }
    }
    float *row = audio + (size_t)voice * (size_t)N;
    if (aligned) {
        *reinterpret_cast<float4 *>(row + n0) = make_float4(o[0], o[1], o[2], o[3]);
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (n0 + i < N) row[n0 + i] = o[i];
    }
}

#ifdef TS_MEASURE
// Measurement aid: the sample loop of the audio kernel (ts_render_run, the same device function) on its own -- no control
// table, no global stores, no CTA turnover, 8 warps per SM sub-partition -- `reps` runs of 20 samples per thread.  What
// the SM pipes can do with this instruction mix: the ALU bound of the audible part.
template <int FASTSIN>
__global__ void __launch_bounds__(1024, 1)
ts_body_bench_kernel(float *__restrict__ sink, int reps, uint32_t nk0, uint32_t nk1, float shape, float tanh_c, uint32_t one_bits,
                     double w0) {
    extern __shared__ __align__(128) float4 bstage[];
    float4 *my = &bstage[threadIdx.x * (TS_RUN / 4)];
    uint2 *my16 = reinterpret_cast<uint2 *>(my);
    nk0 = __reduce_or_sync(0xffffffffu, nk0);  // warp-uniform for the compiler, as blockIdx-derived values are in the real kernel
    nk1 = __reduce_or_sync(0xffffffffu, nk1);
    double P1 = MAGIC32 + 0.1 * threadIdx.x, P2 = (FASTSIN ? MAGIC32 : MAGIC33) + 0.07 * threadIdx.x;
    const double w1 = w0 * (1 + threadIdx.x), w2 = 1.3 * w0 * (1 + threadIdx.x);
#pragma unroll 1
    for (int rep = 0; rep < reps; ++rep) {
        ts_render_run<TS_F32, FASTSIN>(P1, w1, 1e-7, P2, w2, -2e-7, 0.3f, 0.2f, 0.1f, 1e-4f, -1e-4f, 2e-4f,
                                       (uint32_t)(rep * 5 + threadIdx.x * 77 + blockIdx.x), nk0, nk1, shape, tanh_c, one_bits, my, my16);
        P1 += 20.0 * w1;
        P2 += 20.0 * w2;
    }
    __syncthreads();
    float s = 0.f;
    for (int g = 0; g < TS_RUN / 4; ++g) s += my[g].x + my[g].y + my[g].z + my[g].w;
    if (s == 123.456f) sink[threadIdx.x] = s;  // keeps the loop alive; never true in practice
}
#endif  // TS_MEASURE

}  // namespace

#ifdef TS_MEASURE
cudaError_t ts_launch_body_bench(int fastsin, int reps, float *d_sink, cudaStream_t st) {
    static bool attr = false;
    if (!attr) {
        cudaFuncSetAttribute(ts_body_bench_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 1024 * TS_RUN * 4);
        cudaFuncSetAttribute(ts_body_bench_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 1024 * TS_RUN * 4);
        attr = true;
    }
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (fastsin)
        ts_body_bench_kernel<1><<<sms, 1024, 1024 * TS_RUN * 4, st>>>(d_sink, reps, 123u, 456u, 0.4f, 20.f, 0x3f800000u, 1e-3);
    else
        ts_body_bench_kernel<0><<<sms, 1024, 1024 * TS_RUN * 4, st>>>(d_sink, reps, 123u, 456u, 0.4f, 20.f, 0x3f800000u, 1e-3);
    return cudaGetLastError();
}
#endif  // TS_MEASURE

cudaError_t ts_launch_audio_r1(const ts_tick *table, const ts_vhdr *hdr, int B, int64_t N, int K, float *audio, cudaStream_t st) {
    const int64_t gx = (N + 511) / 512;
    if (gx > 0x7fffffffLL || B > 65535) return cudaErrorInvalidValue;
    const int aligned = (N % 4 == 0) && ((reinterpret_cast<uintptr_t>(audio) & 15u) == 0);
    ts_audio_r1_kernel<<<dim3((unsigned)gx, (unsigned)B), 128, 0, st>>>(table, hdr, B, (int)N, K, audio, aligned, 0x3f800000u);
    return cudaGetLastError();
}

cudaError_t ts_launch_audio(const ts_tick *table, const ts_vhdr *hdr, int B, int64_t N, int K, void *audio, int fmt,
                            int mode, int tails, int64_t n_audible_max, double *dbg_phase, cudaStream_t st) {
    const int64_t tiles = (N + TS_TILE - 1) / TS_TILE;
    // two tiles per CTA once the launch is large enough to fill the GPU many times over
    const int tpc = (mode == 0 && tiles * B >= 12000) ? 2 : 1;
    // with TAIL = 1 the silent tiles have no CTA of their own: launch only the tiles that can be audible
    const int64_t tiles_aud = (mode == 0 && tails) ? (n_audible_max + TS_TILE - 1) / TS_TILE : tiles;
    const int64_t tl = (tiles_aud < tiles) ? (tiles_aud > 0 ? tiles_aud : 1) : tiles;
    const int64_t ty = (tl + tpc - 1) / tpc;
    if (ty > 0x7fffffffLL || (ty > 65535 && B > 65535)) return cudaErrorInvalidValue;
    const int swap = ty > 65535;
    const dim3 g = swap ? dim3((unsigned)ty, (unsigned)B) : dim3((unsigned)B, (unsigned)ty);
    // bulk copies and 128-bit stores need 16-byte aligned rows: N a multiple of 4 (fp32) or 8 (16-bit) samples
    const int per16 = (fmt == TS_F32) ? 4 : 8;
    const int aligned = (N % per16 == 0) && ((reinterpret_cast<uintptr_t>(audio) & 15u) == 0);
#define TS_LAUNCH(MODE, TAIL, FMT, TPC) \
    ts_audio_kernel<MODE, TAIL, FMT, TPC><<<g, TS_AUDIO_THREADS, 0, st>>>(table, hdr, B, (int)N, K, audio, dbg_phase, aligned, 0x3f800000u, swap)
#define TS_LAUNCH_T(TAIL, FMT) do { if (tpc == 2) TS_LAUNCH(0, TAIL, FMT, 2); else TS_LAUNCH(0, TAIL, FMT, 1); } while (0)
    if (mode == 0) {
        if (fmt == TS_F32) { if (tails) TS_LAUNCH_T(1, TS_F32); else TS_LAUNCH_T(0, TS_F32); }
        else if (fmt == TS_F16) { if (tails) TS_LAUNCH_T(1, TS_F16); else TS_LAUNCH_T(0, TS_F16); }
        else if (fmt == TS_BF16) { if (tails) TS_LAUNCH_T(1, TS_BF16); else TS_LAUNCH_T(0, TS_BF16); }
        else return cudaErrorInvalidValue;
    } else if (mode == 1) {
        TS_LAUNCH(1, 0, TS_F32, 1);
    } else {
        TS_LAUNCH(2, 0, TS_F32, 1);
    }
#undef TS_LAUNCH_T
#undef TS_LAUNCH
    return cudaGetLastError();
}
