// ts_control.cu -- control-rate stage (S2..S7) and the tick-level phase scan of S9.
//
// 2-D grid over (voice, chunk of 255 control intervals); 256 threads, one control tick each (the last
// thread's tick is the halo shared with the next chunk).  Per tick (tau_j = j*R/sr, S5) a thread evaluates
// the six ADSRs in closed form (S4), the two LFOs (S6; each with its rate and amp ADSR,
// P:L123) and the modulation mixer (S7), all in fp64 because the two pitch rows feed the oscillator phase
// (H1 in DESIGN.md).  The two running sums over time are prefix scans of Q0.64 fixed-point fractions of a
// cycle: __shfl_up_sync inside the warp, per-warp totals inside the CTA, and a decoupled look-back over the
// chunk aggregates of the same voice (each CTA publishes its aggregate with an epoch flag and sums those
// of its predecessors, which always have lower block indices).  Integer addition mod 2^64 is exact and
// associative, so neither the scan order nor the look-back timing can change a bit, and phase does not
// drift however long the render is.
//   * LFO phase  q_j  = q_0 + sum_{i<j} f_i/cr                          (exclusive, mod 1; S6, D21)
//   * VCO phase  Phi_j = phi_0 + sum_{i<j} S_i, S_i = sum of the R increments of interval i.
//     Inside an interval pitch is linear in n (S8), so the increments are a geometric sequence:
//     S_i = inc_i * (1 + rho + ... + rho^(R-1)), built by doubling (no division, no singularity at rho = 1).
// The audio kernel then needs nothing from other threads: every run of 20 samples starts from the
// table entry of its tick.
#include "ts_common.cuh"
#include "ts_math.cuh"

// Both tables live in GLOBAL memory: every thread reads its own entry, which the constant cache would serialise
// (one distinct address per cycle; it showed up as 34 % ADU-pipe load), while LDG coalesces it.
struct ts_range_dev {
    double lo, hi, curve, inv_curve;  // inv_curve = 1 / curve, divided once on the host (IEEE: same bits as here)
    long long symmetric;
};
__device__ ts_range_dev c_nebula[TS_NPARAM];
__device__ ts_math_tables c_math;

cudaError_t ts_upload_nebula(const ts_range *host78, cudaStream_t st) {
    static ts_range_dev D[TS_NPARAM];  // static: the async copy reads it after this function returns
    ts_nebula_to_device_layout(host78, D);
    return cudaMemcpyToSymbolAsync(c_nebula, D, sizeof D, 0, cudaMemcpyHostToDevice, st);
}
size_t ts_nebula_device_bytes() { return sizeof(ts_range_dev) * TS_NPARAM; }
void ts_nebula_to_device_layout(const ts_range *host78, void *out) {
    ts_range_dev *D = static_cast<ts_range_dev *>(out);
    for (int i = 0; i < TS_NPARAM; ++i)
        D[i] = ts_range_dev{host78[i].lo, host78[i].hi, host78[i].curve, 1.0 / host78[i].curve, (long long)host78[i].symmetric};
}

cudaError_t ts_upload_math_tables(cudaStream_t st) {
    static ts_math_tables T;  // static: the async copy reads it after this function returns
    for (int i = 0; i < TS_LOG_N; ++i) {
        const unsigned long long lo = TS_LOG_OFF + ((unsigned long long)i << 47), hi = lo + (1ull << 47);
        double zlo, zhi;
        memcpy(&zlo, &lo, 8);
        memcpy(&zhi, &hi, 8);
        const long double c = ((long double)zlo + (long double)zhi) / 2.0L;
        T.invc[i] = (double)(1.0L / c);
        T.logc[i] = (double)(-log2l((long double)T.invc[i]));
    }
    for (int i = 0; i < TS_EXP_N; ++i) T.exp2t[i] = (double)exp2l((long double)i / TS_EXP_N);
    return cudaMemcpyToSymbolAsync(c_math, &T, sizeof T, 0, cudaMemcpyHostToDevice, st);
}

// S3 map(u; lo,hi,c,S).  __dmul_rn/__dadd_rn: one rounding per operation (no FMA contraction), so the
// affine parameters come out bit-identical to a plain IEEE evaluation of the same expression.
__device__ __noinline__ double ts_pow_slow(double x, double a) { return pow(x, a); }  // cold paths only

// x^a for x in [0,1], a > 0, exact at both ends
__device__ __forceinline__ double ts_pow_unit(double x, double a, const ts_math_tables *T) {
    if (x <= 0.0) return 0.0;
    if (x >= 1.0) return 1.0;
    return ts_pow01(x, a, T);
}

__device__ __forceinline__ double ts_map(double u, const ts_range_dev &r, const ts_math_tables *T) {
    if (!(u >= 0.0)) u = 0.0;
    if (u > 1.0) u = 1.0;
    if (!r.symmetric) {
        const double v = (r.curve == 1.0) ? u : ts_pow_unit(u, r.inv_curve, T);
        return __dadd_rn(r.lo, __dmul_rn(r.hi - r.lo, v));
    }
    const double d = __dadd_rn(__dmul_rn(2.0, u), -1.0);
    const double a = fabs(d);
    const double v = (r.curve == 1.0) ? a : ts_pow_unit(a, r.inv_curve, T);
    const double s = (d > 0.0) ? 1.0 : ((d < 0.0) ? -1.0 : 0.0);
    return __dadd_rn((r.lo + r.hi) / 2.0, __dmul_rn((r.hi - r.lo) / 2.0, s * v));
}


// S4 ramp(t,s,d)^alpha.  pow(0,a) = 0 and pow(1,a) = 1 exactly for a > 0, so the saturated ends skip pow.
// The saturation tests are the oracle's own comparisons (exact); inside the ramp x/d is x * (1/d).
__device__ __forceinline__ double ts_ramp_pow(double t, double s, double d, double invd, double alpha,
                                              const ts_math_tables *T) {
    const double x = t - s;
    if (!(alpha > 0.0)) return ts_pow_slow((x >= d) ? 1.0 : ((x <= 0.0) ? 0.0 : x / d), alpha);  // not with alpha > 0
    if (x >= d) return 1.0;
    if (x <= 0.0) return 0.0;
    const double r = x * invd;
    return (r >= 1.0) ? 1.0 : ts_pow01(r, alpha, T);
}

// E(t) = ramp(t,0,A)^a * [1 - (1-S) ramp(t,A,Dc)^a] * [1 - ramp(t,D,Rl)^a];  V ramps ordered release, attack, decay
__device__ __forceinline__ double ts_adsr(double t, int e, const ts_voice_consts &V, const ts_math_tables *T) {
    const double S = V.h[4 + 5 * e], al = V.h[6 + 5 * e];
    const double *rs = &V.rs[3 * e], *rd = &V.rd[3 * e], *ri = &V.rinv[3 * e];
    const double r = ts_ramp_pow(t, rs[0], rd[0], ri[0], al, T);
    if (r == 1.0) return 0.0;  // a * (...) * (1 - 1) = 0 exactly
    const double a = ts_ramp_pow(t, rs[1], rd[1], ri[1], al, T);
    if (a == 0.0) return 0.0;
    const double d = ts_ramp_pow(t, rs[2], rd[2], ri[2], al, T);
    return a * (1.0 - (1.0 - S) * d) * (1.0 - r);
}

// x^a for x in [0,1], a > 0, without branches: exact 0 and 1 at the ends (S4 needs both: E = 0 exactly once the
// release is over), clamped log2/exp2 in between.  Twelve of these per tick are independent chains, so the
// fp64 latency that dominates this kernel overlaps instead of adding up.
// x comes from ts_ramp_lin, i.e. it is already in [0, 1]; x = 0 needs no clamp either: ts_log2 works on the bit pattern and
// returns about -1023 for it, the product is clamped to -1000 and the result is replaced by the exact 0 below.
__device__ __forceinline__ double ts_pow01_sel(double x, double a, const ts_math_tables *T) {
    double p = ts_exp2(fmax(a * ts_log2(x, T), -1000.0), T);
    p = (x >= 1.0) ? 1.0 : p;
    return (x <= 0.0) ? 0.0 : p;
}
__device__ __forceinline__ double ts_ramp_lin(double t, double s, double d, double invd) {  // S4 ramp(t,s,d)
    const double x = t - s;
    return (x >= d) ? 1.0 : ((x <= 0.0) ? 0.0 : x * invd);
}
// Same E(t) as ts_adsr for alpha > 0.  While the attack ramp is below 1 the decay ramp is 0 and afterwards the
// attack ramp is 1, so ONE power serves both: two powers per envelope instead of three.
__device__ __forceinline__ double ts_adsr_fast(double t, int e, const ts_voice_consts &V, const ts_math_tables *T) {
    const double S = V.h[4 + 5 * e], al = V.h[6 + 5 * e];
    const double *rs = &V.rs[3 * e], *rd = &V.rd[3 * e], *ri = &V.rinv[3 * e];
    const double r = ts_ramp_lin(t, rs[0], rd[0], ri[0]);
    const double a = ts_ramp_lin(t, rs[1], rd[1], ri[1]);
    const double d = ts_ramp_lin(t, rs[2], rd[2], ri[2]);
    const bool in_attack = a < 1.0;
    const double m = in_attack ? a : d;
    // A power is evaluated only if some lane of the warp is strictly inside that ramp (32 consecutive ticks = 73 ms:
    // during sustain, before the note-off and after the release nothing is).  Called by full warps only.
    double pm = (m >= 1.0) ? 1.0 : 0.0, pr = (r >= 1.0) ? 1.0 : 0.0;
    if (__any_sync(0xffffffffu, m > 0.0 && m < 1.0)) pm = ts_pow01_sel(m, al, T);
    if (__any_sync(0xffffffffu, r > 0.0 && r < 1.0)) pr = ts_pow01_sel(r, al, T);
    const double pa = in_attack ? pm : 1.0, pd = in_attack ? 0.0 : pm;
    return pa * (1.0 - (1.0 - S) * pd) * (1.0 - pr);
}

// frac of a double as Q0.64
__device__ __forceinline__ unsigned long long ts_frac_q64(double x) {
    const double f = x - floor(x);  // exact, in [0,1)
    return __double2ull_rz(f * 18446744073709551616.0);
}
__device__ __forceinline__ double ts_q64_to_double(unsigned long long q) {
    return __ull2double_rz(q >> 11) * (1.0 / 9007199254740992.0);  // exact truncation to 53 bits, [0,1)
}

// Block-wide exclusive scan (mod 2^64) of two values per thread, in thread order: __shfl_up_sync inside
// the warp, per-warp totals through shared memory.  sm: 64 words of scratch.
__device__ __forceinline__ void ts_block_scan2(unsigned long long &a, unsigned long long &b, unsigned long long *sm) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    unsigned long long ia = a, ib = b;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long ua = __shfl_up_sync(0xffffffffu, ia, o);
        const unsigned long long ub = __shfl_up_sync(0xffffffffu, ib, o);
        if (lane >= o) { ia += ua; ib += ub; }
    }
    if (lane == 31) { sm[wid] = ia; sm[32 + wid] = ib; }
    __syncthreads();
    unsigned long long oa = 0, ob = 0;
    for (int w = 0; w < wid && w < nw; ++w) { oa += sm[w]; ob += sm[32 + w]; }  // <= 7 terms for 256 threads
    a = oa + ia - a;
    b = ob + ib - b;
    __syncthreads();  // scratch may be reused
}

#ifndef TS_CTL_THREADS_N
#define TS_CTL_THREADS_N 256
#endif
constexpr int TS_CTL_THREADS = TS_CTL_THREADS_N;  // 255 control intervals per chunk: 128 / 256 / 512 measured 32.9 / 32.4 / 32.5 us per C2 step, 64 worse
constexpr int TS_SETUP_THREADS = 128;  // the setup kernel's thread roles are laid out for 128 threads
constexpr int TS_CTL_IC = TS_CTL_THREADS - 1;  // control intervals per chunk (the last thread is the halo tick)

// ---- decoupled look-back over the chunk aggregates of one voice ------------------------------------
// A slot is two 16-byte words, each a Q0.64 sum with the launch epoch beside it: one 128-bit store publishes a word,
// one 128-bit load reads value and flag together (aligned 16-byte accesses are single transactions), so neither side
// needs a fence -- the same packing CUB's single-word tile descriptors use.
// What this rests on (reading D28): (i) an aligned 16-byte volatile vector access is ONE memory transaction on
// sm_100, so value and epoch are never seen half-written -- the PTX memory model itself only promises this per scalar
// element; (ii) a CTA with a lower linear block index has been dispatched before this one.  (i) is checked, not trusted:
// the epoch is written into BOTH trailing 32-bit fields of a word (the two ends of the 16 bytes a torn access could
// split), and a reader takes a word only when both equal the launch epoch -- a torn read spins again instead of being
// summed.  (ii) cannot be checked from inside; its failure mode is the bounded spin below (TS_ECUDA at the next ts_sync).
struct __align__(16) ts_agg_word {
    unsigned long long s;
    unsigned int flag;   // == launch epoch once s is valid
    unsigned int flag2;  // the same epoch again
};
struct __align__(16) ts_agg {
    ts_agg_word w[2];
};
static_assert(sizeof(ts_agg) == 32, "ts_agg layout");

__device__ __forceinline__ void ts_publish(ts_agg *slot, unsigned long long a, unsigned long long b, unsigned int epoch) {
    uint4 w0, w1;
    w0.x = (unsigned int)a; w0.y = (unsigned int)(a >> 32); w0.z = epoch; w0.w = epoch;
    w1.x = (unsigned int)b; w1.y = (unsigned int)(b >> 32); w1.z = epoch; w1.w = epoch;
    asm volatile("st.volatile.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(&slot->w[0]), "r"(w0.x), "r"(w0.y), "r"(w0.z), "r"(w0.w) : "memory");
    asm volatile("st.volatile.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(&slot->w[1]), "r"(w1.x), "r"(w1.y), "r"(w1.z), "r"(w1.w) : "memory");
}
// A predecessor always has a lower linear block index, so it has been dispatched before this CTA (in-order dispatch);
// the wait is nevertheless bounded: after TS_SPIN_LIMIT polls (about a second) the thread raises the launch's error
// flag and goes on with what it has, and the host turns the flag into TS_ECUDA at the next ts_sync().
constexpr int TS_SPIN_LIMIT = 1 << 24;
__device__ __forceinline__ void ts_wait_slot(const ts_agg *p, unsigned int epoch, unsigned int *err, unsigned long long &a,
                                             unsigned long long &b) {
    uint4 v0, v1;
    int spins = 0;
    for (;;) {  // both words in flight at once: one L2 round trip when the predecessor has already published
        asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v0.x), "=r"(v0.y), "=r"(v0.z), "=r"(v0.w) : "l"(&p->w[0]) : "memory");
        asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v1.x), "=r"(v1.y), "=r"(v1.z), "=r"(v1.w) : "l"(&p->w[1]) : "memory");
        if (v0.z == epoch && v0.w == epoch && v1.z == epoch && v1.w == epoch) break;
        __nanosleep(40);
        if (++spins > TS_SPIN_LIMIT) {
            atomicExch(err, 1u);
            break;
        }
    }
    a = ((unsigned long long)v0.y << 32) | v0.x;
    b = ((unsigned long long)v1.y << 32) | v1.x;
}
// Sum of the aggregates of chunks 0 .. c-1 (mod 2^64): every thread fetches its share of the predecessors, the partial
// sums meet through warp shuffles and one shared-memory word per warp.  Call with all threads; the totals are in
// sm[0 .. nw) and sm[32 .. 32 + nw) after the caller's next __syncthreads().
__device__ __forceinline__ void ts_lookback(const ts_agg *slots, int c, unsigned int epoch, unsigned long long *sm /*[64]*/,
                                            unsigned int *err) {
    unsigned long long a = 0ull, b = 0ull;
    if ((int)(threadIdx.x & ~31u) < c) {  // warps without a predecessor to fetch skip the reduction
        for (int i = threadIdx.x; i < c; i += blockDim.x) {
            unsigned long long x, y;
            ts_wait_slot(&slots[i], epoch, err, x, y);
            a += x;
            b += y;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_down_sync(0xffffffffu, a, o);
            b += __shfl_down_sync(0xffffffffu, b, o);
        }
    }
    if ((threadIdx.x & 31) == 0) {
        sm[threadIdx.x >> 5] = a;
        sm[32 + (threadIdx.x >> 5)] = b;
    }
}
__device__ __forceinline__ void ts_lookback_total(const unsigned long long *sm, int c, unsigned long long &a, unsigned long long &b) {
    a = sm[0];
    b = sm[32];
    if (c > 32) {  // more than one warp fetched predecessors
#pragma unroll
        for (int w = 1; w < TS_CTL_THREADS / 32; ++w) {
            a += sm[w];
            b += sm[32 + w];
        }
    }
}

// S6 LFO value at phase p in [0,1): blend of the five shapes with pre-normalised weights (D11).
// sin(2 pi p) for p in [0,1) without branches: y = 2p - 1, sin(2 pi p) = -sin(pi y); |y| > 1/2 is folded back with
// sin(pi - x) = sin x, then the Taylor series of sin(pi y) to y^19 (truncation 2.6e-16 at |y| = 1/2).
__device__ __forceinline__ double ts_sin2pi(double p) {
    double y = 2.0 * p - 1.0;
    y = (fabs(y) > 0.5) ? copysign(1.0, y) - y : y;
    const double y2 = y * y;
    double q = c_coef.sin2pip[9];
#pragma unroll
    for (int k = 8; k >= 0; --k) q = fma(q, y2, c_coef.sin2pip[k]);
    return -(q * y);
}

__device__ __forceinline__ double ts_lfo_mix(double p, const double *wn) {
    const double t = p + 0.75;
    double v = wn[0] * ts_sin2pi(p);
    v = fma(wn[1], 4.0 * fabs((t - floor(t)) - 0.5) - 1.0, v);
    v = fma(wn[2], 2.0 * p - 1.0, v);
    v = fma(wn[3], 1.0 - 2.0 * p, v);
    v = fma(wn[4], (p < 0.5) ? 1.0 : -1.0, v);
    return v;
}


// ---- per-voice setup: one CTA per voice ----------------------------------------------------------------------------
// S1 (optional: the fused sampler of the streaming path), S2/S3 parameter map, the constants every tick needs, the
// first tick at which the voice is silent for good, and the voice header of the audio kernel.  Everything here used to
// be recomputed by every chunk CTA of the control kernel (2.3 us each); now it runs once per voice.
__global__ void __launch_bounds__(TS_SETUP_THREADS)
ts_setup_kernel(ts_voice *__restrict__ params, int sample, uint64_t seed, uint64_t g0, int B, int sr, int R, long long N, int K,
                ts_voice_consts *__restrict__ vc, ts_vhdr *__restrict__ hdr, float *__restrict__ params_human,
                unsigned long long *__restrict__ d_active, int full, const ts_range_dev *__restrict__ neb_table) {
    const ts_range_dev *neb = neb_table ? neb_table : c_nebula;  // a table of this launch's own (per-batch nebulae) or the active one
    __shared__ ts_voice_consts V;
    __shared__ ts_math_tables MT;
    __shared__ __align__(16) float su[TS_NPARAM + 2];
    __shared__ uint32_t s_nk[2];
    __shared__ float s_tanh_c;
    __shared__ int s_fast;
    const int tid = threadIdx.x, v = blockIdx.x;
    if (tid < (int)(sizeof(ts_math_tables) / 8))  // table look-ups from shared memory: ~30 cycles instead of an L2 round trip each
        reinterpret_cast<double *>(&MT)[tid] = reinterpret_cast<const double *>(&c_math)[tid];
    if (sample) {  // S1: Philox blocks 0..19 carry the parameters, thread 20 draws the noise key (D4)
        const uint64_t g = g0 + (uint64_t)v;
        const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
        if (tid < 20) {
            uint32_t w[4];
            ts_philox4x32_10((uint32_t)tid, (uint32_t)g, (uint32_t)(g >> 32), 0u, k0, k1, w);
#pragma unroll
            for (int i = 0; i < 4; ++i) su[4 * tid + i] = (float)(w[i] >> 8) * (1.0f / 16777216.0f);
        } else if (tid == 20) {
            uint32_t nk[4];
            ts_philox4x32_10(0u, (uint32_t)g, (uint32_t)(g >> 32), 2u, k0, k1, nk);
            s_nk[0] = nk[0];
            s_nk[1] = nk[1];
        }
        __syncthreads();
        if (tid < 20) {  // the record: u[78] then the two key words, 16 bytes per thread
            float4 r = *reinterpret_cast<const float4 *>(&su[4 * tid]);
            if (tid == 19) { r.z = __uint_as_float(s_nk[0]); r.w = __uint_as_float(s_nk[1]); }
            reinterpret_cast<float4 *>(params + v)[tid] = r;
        }
    } else {
        if (tid < TS_NPARAM) su[tid] = params[v].u[tid];
        if (tid < 2) s_nk[tid] = params[v].noise_key[tid];
        __syncthreads();
    }
    if (tid < TS_NPARAM) {
        const double hv = ts_map((double)su[tid], neb[tid], &MT);
        V.h[tid] = hv;
        if (params_human) params_human[(size_t)v * TS_NPARAM + tid] = (float)hv;
    }
    __syncthreads();
    const double *h = V.h;
    const double D = h[1];
    const double cr = (double)sr / (double)R;  // control rate (D2): one tick every R samples
    if (tid < 18) {  // ramps of ADSR e: release (starts at D), attack (0), decay (A)
        const int e = tid / 3, k = tid - 3 * e;
        const double A = h[2 + 5 * e], Dc = h[3 + 5 * e], Rl = h[5 + 5 * e];
        const double st = (k == 0) ? D : ((k == 1) ? 0.0 : A), d = (k == 0) ? Rl : ((k == 1) ? A : Dc);
        V.rs[tid] = st;
        V.rd[tid] = d;
        V.rinv[tid] = (d > 0.0) ? 1.0 / d : 0.0;
    } else if (tid >= 32 && tid < 42) {
        const int l = (tid - 32) / 5, i = (tid - 32) - 5 * l;
        const double *w = &h[35 + 8 * l];
        const double den = (((w[0] + w[1]) + w[2]) + w[3]) + w[4];
        V.lfo_w[l][i] = (den == 0.0) ? 0.0 : w[i] / den;
    } else if (tid >= 42 && tid < 46) {
        const int l = (tid - 42) & 1;
        if (tid < 44) V.dq_f[l] = h[32 + 8 * l] / cr;
        else V.dq_d[l] = h[33 + 8 * l] / cr;
    } else if (tid >= 64 && tid < 84) {
        const int d = (tid - 64) >> 2, sidx = (tid - 64) & 3;
        const double *w = &h[48 + 4 * d];
        const double den = ((w[0] + w[1]) + w[2]) + w[3];
        V.mix_w[d][sidx] = (den == 0.0) ? 0.0 : w[sidx] / den;
    } else if (tid >= 46 && tid < 49) {
        const int i = tid - 46;
        const double lsum = (h[75] + h[76]) + h[77];
        const double gi = (lsum == 0.0) ? 0.0 : h[75 + i] / lsum;
        V.g[i] = (i == 1) ? gi * (1.0 - h[74] / 2.0) : gi;  // VCO2 carries (1 - s/2) of S11
    } else if (tid == 50) {  // S11: steepness of the square/saw from the unmodulated note frequency, as the tanh constant
        const double fc = 440.0 * ts_exp2((h[0] + h[71] - 69.0) * (1.0 / 12.0), &MT);
        const double k = 12000.0 / (fc * (ts_log2(fc, &MT) * 0.30102999566398120));
        s_tanh_c = (float)(1.5707963267948966 * k * 2.0 * 1.4426950408889634);
        s_fast = (k <= 512.0) ? 1 : 0;  // ts_audio.cu: whole-cycle MUFU.SIN / MUFU.COS variant of the square/saw
    } else if (tid >= 96) {
        // The voice is silent for good once the release of all four audible envelopes is over (their
        // ramp is 1, so E = 0 exactly): adsr1, adsr2, lfo1_amp, lfo2_amp.  jsil = first tick with
        // (tau - D) >= rl_max, evaluated exactly as S4's ramp does; the predicate is monotone in j, so the 32 lanes
        // of this warp test 32 candidates around the estimate at once (one fp64 division each, not a serial walk).
        const double rl_max = fmax(fmax(h[2 + 3], h[7 + 3]), fmax(h[12 + 3], h[22 + 3]));
        const int lane = tid - 96;
        long long je = (long long)floor((D + rl_max) * cr) - 8;
        if (je > K) je = K;
        if (je < 0) je = 0;
        auto silent_at = [&](long long jj) { return jj >= K || (((double)(jj * R) / (double)sr) - D >= rl_max); };
        const unsigned int hit = __ballot_sync(0xffffffffu, silent_at(je + lane));
        long long j = hit ? je + (__ffs(hit) - 1) : je + 32;
        if (lane == 0 && (hit & 1u)) {  // estimate off (cannot happen for finite parameters): walk
            while (j > 0 && silent_at(j - 1)) --j;
        } else if (lane == 0 && !hit) {
            while (!silent_at(j)) ++j;
        }
        j = __shfl_sync(0xffffffffu, j, 0);
        if (tid == 96) {
            if (full) j = K;  // debug exports: evaluate every tick
            V.jsil = (int)j;
            int slow = 0;
            for (int e = 0; e < 6; ++e) slow |= !(h[6 + 5 * e] > 0.0);
            V.slow = slow;
            V.pad[0] = V.pad[1] = 0;
        }
    }
    __syncthreads();
    if (tid < (int)(sizeof(ts_voice_consts) / 16))
        reinterpret_cast<uint4 *>(vc + v)[tid] = reinterpret_cast<const uint4 *>(&V)[tid];
    if (tid == 96) {  // the voice header of the audio kernel
        const long long j = V.jsil;
        const long long n_act = (j * R < N) ? j * R : N;
        ts_vhdr hd;
        hd.shape = (float)h[74];
        hd.tanh_c = s_tanh_c;
        hd.nk0 = s_nk[0];
        hd.nk1 = s_nk[1];
        hd.n_act = (int32_t)n_act;
        hd.n_ticks = (int32_t)((j + 1 < K) ? j + 1 : K);
        hd.pad[0] = s_fast;
        hd.pad[1] = 0;
        hdr[v] = hd;
        if (d_active) atomicAdd(d_active, (unsigned long long)n_act);
    }
}

// PHASES = 1: controls + the S9 tick-level phase scan + the control table of the audio kernel (R = TS_R);
// PHASES = 2: the same for the audio-rate-control mode R = 1 (an interval is one sample: its phase advance is the
//             increment itself, no geometric sums);
// PHASES = 0: stops after the modulation mixer (control-rate rendering on its own: no interval sums, no second scan)
template <int PHASES>
__global__ void __launch_bounds__(TS_CTL_THREADS)
ts_control_kernel(const ts_voice_consts *__restrict__ vc, int B, int sr, int R, long long N, int K, int NC,
                  ts_tick *__restrict__ table, ts_agg *__restrict__ agg, unsigned int epoch, double *__restrict__ dbg_ctl,
                  unsigned int *__restrict__ err, int swap, long long J, double f0) {
    __shared__ ts_voice_consts V;
    __shared__ ts_math_tables MT;
    __shared__ unsigned long long scan_sm[64];
    __shared__ unsigned long long lb_sm[64];
    __shared__ double2 pitch[TS_CTL_THREADS];
    __shared__ double Es[6][TS_CTL_THREADS];

    const int tid = threadIdx.x;
    // 2-D grid, no integer division (x = voice, y = chunk; swapped when a voice has more than 65535 chunks): either way
    // a chunk's predecessors have lower linear block indices
    const int c = swap ? blockIdx.x : blockIdx.y, v = swap ? blockIdx.y : blockIdx.x;
    const int j0 = c * TS_CTL_IC;
    const int jsil = vc[v].jsil;
    if (c > 0 && j0 >= jsil) {  // nothing audible from this chunk on (55 % of C2's chunks); no successor waits for it
        if (dbg_ctl) {            // control-rate rendering: ticks after the voice has gone silent are 0
            // ticks j0 + 1 .. j0 + 126, plus the first tick if the previous chunk is dead too (a live one writes its halo)
            const int j = j0 + tid;
            const bool prev_live = (c == 1) || (j0 - TS_CTL_IC < jsil);
            if (tid < TS_CTL_IC && (tid > 0 || !prev_live) && j < K) {
                double *o = dbg_ctl + (size_t)v * 5 * K;
#pragma unroll
                for (int d = 0; d < 5; ++d) o[(size_t)d * K + j] = 0.0;
            }
        }
        return;
    }
    ts_tick *tab = table + (size_t)v * K;
    ts_agg *agg_q = agg + ((size_t)v * NC) * 2, *agg_p = agg_q + NC;

    // ---- stage the math tables and the voice's constants ----
    for (int i = tid; i < (int)(sizeof(ts_math_tables) / 8); i += TS_CTL_THREADS)
        reinterpret_cast<double *>(&MT)[i] = reinterpret_cast<const double *>(&c_math)[i];
    for (int i = tid; i < (int)(sizeof(ts_voice_consts) / 16); i += TS_CTL_THREADS)
        reinterpret_cast<uint4 *>(&V)[i] = __ldg(reinterpret_cast<const uint4 *>(vc + v) + i);
    __syncthreads();
    const double *h = V.h;
    // J = ceil(N / R): control intervals that hold samples; f0 = 440 / sr: both divided once on the host

    // ================= phase 1: controls at tick j =================
    const int j = j0 + tid;
    const bool live = (j <= jsil) && (j < K);
    double E[6] = {0, 0, 0, 0, 0, 0};
    unsigned long long dq1 = 0, dq2 = 0;
    const double tau = (double)((long long)j * R) / (double)sr;
    if (V.slow) {  // some alpha <= 0 (custom nebula): generic path, uniform over the voice
        if (live) {
#pragma unroll 1
            for (int e = 0; e < 6; ++e) Es[e][tid] = ts_adsr(tau, e, V, &MT);
#pragma unroll
            for (int e = 0; e < 6; ++e) E[e] = Es[e][tid];
        }
    } else if (j0 + (tid & ~31) <= jsil) {  // warps with a live lane, every lane of them (the warp votes on which powers are
                                            // needed at all; dead lanes' values are unused); unrolled: partial unrolling measured slower
#pragma unroll
        for (int e = 0; e < 6; ++e) E[e] = ts_adsr_fast(tau, e, V, &MT);
    }
    if (live) {
        const double d1 = fma(V.dq_d[0], E[3], V.dq_f[0]);
        const double d2 = fma(V.dq_d[1], E[5], V.dq_f[1]);
        dq1 = (unsigned long long)__double2ll_rn((d1 - rint(d1)) * 18446744073709551616.0);
        dq2 = (unsigned long long)__double2ll_rn((d2 - rint(d2)) * 18446744073709551616.0);
    }
    ts_block_scan2(dq1, dq2, scan_sm);  // exclusive prefix inside the chunk
    if (tid == TS_CTL_IC) ts_publish(&agg_q[c], dq1, dq2, epoch);  // halo thread: sum over the chunk's own ticks
    ts_lookback(agg_q, c, epoch, lb_sm, err);
    __syncthreads();
    unsigned long long lbq1, lbq2;
    ts_lookback_total(lb_sm, c, lbq1, lbq2);
    const unsigned long long q1 = ts_frac_q64(h[34]) + lbq1 + dq1, q2 = ts_frac_q64(h[42]) + lbq2 + dq2;
    // the halo tick is written by the next chunk unless that chunk has nothing to do
    const bool own = (tid < TS_CTL_IC) || (j0 + TS_CTL_IC >= jsil) || (c == NC - 1);
    double M[5] = {0, 0, 0, 0, 0};
    if (live) {
        const double L1 = E[2] * ts_lfo_mix(ts_q64_to_double(q1), V.lfo_w[0]);
        const double L2 = E[4] * ts_lfo_mix(ts_q64_to_double(q2), V.lfo_w[1]);
#pragma unroll
        for (int d = 0; d < 5; ++d)
            M[d] = fma(V.mix_w[d][3], L2, fma(V.mix_w[d][2], L1, fma(V.mix_w[d][1], E[1], V.mix_w[d][0] * E[0])));
        if (PHASES) {
            pitch[tid] = make_double2(fma(h[69], M[0], h[0] + h[68]), fma(h[72], M[2], h[0] + h[71]));
            if (own) {
                float4 a;
                a.x = (float)(M[1] * V.g[0]);
                a.y = (float)(M[3] * V.g[1]);
                a.z = (float)(M[4] * V.g[2]);
                a.w = 0.0f;
                *reinterpret_cast<float4 *>(&tab[j].a1) = a;
            }
        }
    }
    if (dbg_ctl && own && j < K) {  // ticks after the voice has gone silent for good are 0
        double *o = dbg_ctl + (size_t)v * 5 * K;
#pragma unroll
        for (int d = 0; d < 5; ++d) o[(size_t)d * K + j] = M[d];
    }
    if (!PHASES) return;
    __syncthreads();

    // ================= phase 2: interval j (pitch is linear between ticks j and j+1) =================
    const bool act = (tid < TS_CTL_IC) && (j < jsil) && (j < J);
    unsigned long long s1 = 0, s2 = 0;
    double inc[2] = {0, 0}, e1[2] = {0, 0}, g20[2] = {TS_RUN, TS_RUN};
    if (act) {
        const double2 p0 = pitch[tid], p1 = pitch[tid + 1];
#pragma unroll 1
        for (int o = 0; o < 2; ++o) {
            const double pa = o ? p0.y : p0.x, pb = o ? p1.y : p1.x;
            const double inc0_ = f0 * ts_exp2((pa - 69.0) * (1.0 / 12.0), &MT);
            if (PHASES == 2) {  // R = 1: the interval holds one sample
                const unsigned long long sf1 = ts_frac_q64(inc0_);
                if (o) { s2 = sf1; inc[1] = inc0_; e1[1] = 0.0; g20[1] = 1.0; }
                else   { s1 = sf1; inc[0] = inc0_; e1[0] = 0.0; g20[0] = 1.0; }
                continue;
            }
            const double x1 = ts_expm1_small((pb - pa) * (0.69314718055994530942 / (12.0 * TS_R)));  // rho - 1
            // geometric sums by doubling: x_m = rho^m - 1, g_m = 1 + rho + ... + rho^(m-1)
            const double x2 = x1 * (2.0 + x1), x4 = x2 * (2.0 + x2);
            const double g2 = 2.0 + x1, g4 = g2 * (2.0 + x2);
            const double g5 = g4 + (1.0 + x4), x5 = fma(x4, x1, x4 + x1);
            const double g10 = g5 * (2.0 + x5), x10 = x5 * (2.0 + x5);
            const double g20_ = g10 * (2.0 + x10), x20 = x10 * (2.0 + x10);
            const double g40 = g20_ * (2.0 + x20), x40 = x20 * (2.0 + x20);
            const double g80 = g40 * (2.0 + x40), x80 = x40 * (2.0 + x40);
            const double g100 = fma(1.0 + x80, g20_, g80);
            const double inc_ = inc0_;
            const unsigned long long sf = ts_frac_q64(inc_ * g100);
            if (o) { s2 = sf; inc[1] = inc_; e1[1] = x1; g20[1] = g20_; }
            else   { s1 = sf; inc[0] = inc_; e1[0] = x1; g20[0] = g20_; }
        }
    }
    ts_block_scan2(s1, s2, scan_sm);
    if (tid == TS_CTL_IC) ts_publish(&agg_p[c], s1, s2, epoch);
    ts_lookback(agg_p, c, epoch, lb_sm, err);
    __syncthreads();
    if (act) {
        unsigned long long lbp1, lbp2;
        ts_lookback_total(lb_sm, c, lbp1, lbp2);
        const unsigned long long P1 = ts_frac_q64(h[70]) + lbp1 + s1, P2 = ts_frac_q64(h[73]) + lbp2 + s2;
        double2 *d2 = reinterpret_cast<double2 *>(&tab[j]);
        d2[0] = make_double2(ts_q64_to_double(P1), inc[0]);
        d2[1] = make_double2(e1[0], g20[0]);
        d2[2] = make_double2(ts_q64_to_double(P2), inc[1]);
        d2[3] = make_double2(e1[1], g20[1]);
    }
}

size_t ts_control_agg_bytes(int B, int K) {
    const int J = K - 1, NC = (J + TS_CTL_IC - 1) / TS_CTL_IC > 0 ? (J + TS_CTL_IC - 1) / TS_CTL_IC : 1;
    return (size_t)B * NC * 2 * sizeof(ts_agg);
}

cudaError_t ts_launch_setup(ts_voice *d_params, int sample, uint64_t seed, uint64_t g0, int B, int sr, int R, int64_t N, int K,
                            ts_voice_consts *vc, ts_vhdr *hdr, float *params_human, unsigned long long *d_active, int full,
                            const void *d_nebula, cudaStream_t st) {
    ts_setup_kernel<<<(unsigned)B, TS_SETUP_THREADS, 0, st>>>(d_params, sample, seed, g0, B, sr, R, (long long)N, K, vc, hdr,
                                                          params_human, d_active, full, static_cast<const ts_range_dev *>(d_nebula));
    return cudaGetLastError();
}

cudaError_t ts_launch_control(const ts_voice_consts *vc, int B, int sr, int R, int64_t N, int K, ts_tick *table, void *agg,
                              unsigned int epoch, double *dbg_ctl, int phases, int64_t n_audible_max, unsigned int *d_err, cudaStream_t st) {
    const int J = K - 1;
    int NC = (J + TS_CTL_IC - 1) / TS_CTL_IC;
    if (NC < 1) NC = 1;
    // chunks that start at or after the last tick any voice can be audible at are dead for every voice: not launched
    // (unless the caller wants the zeros of the control-rate output written, or every tick evaluated)
    int NCL = NC;
    if (!dbg_ctl && n_audible_max >= 0) {
        const int64_t jmax = (n_audible_max + R - 1) / R + 1;
        const int64_t need = (jmax + TS_CTL_IC - 1) / TS_CTL_IC;
        if (need < NCL) NCL = (int)(need > 0 ? need : 1);
    }
    if (NCL > 65535 && B > 65535) return cudaErrorInvalidValue;
    const int swap = NCL > 65535;
    const dim3 grid = swap ? dim3((unsigned)NCL, (unsigned)B) : dim3((unsigned)B, (unsigned)NCL);
    if (phases && R != TS_R && R != 1) return cudaErrorInvalidValue;  // the audio kernels are built on R = 100 and R = 1
    const long long J64 = ((long long)N + R - 1) / R;
    const double f0 = 440.0 / (double)sr;
    if (phases && R == 1)
        ts_control_kernel<2><<<grid, TS_CTL_THREADS, 0, st>>>(vc, B, sr, R, (long long)N, K, NC, table,
                                                             static_cast<ts_agg *>(agg), epoch, dbg_ctl, d_err, swap, J64, f0);
    else if (phases)
        ts_control_kernel<1><<<grid, TS_CTL_THREADS, 0, st>>>(vc, B, sr, R, (long long)N, K, NC, table,
                                                                       static_cast<ts_agg *>(agg), epoch, dbg_ctl, d_err, swap, J64, f0);
    else
        ts_control_kernel<0><<<grid, TS_CTL_THREADS, 0, st>>>(vc, B, sr, R, (long long)N, K, NC, table,
                                                                       static_cast<ts_agg *>(agg), epoch, dbg_ctl, d_err, swap, J64, f0);
    return cudaGetLastError();
}
