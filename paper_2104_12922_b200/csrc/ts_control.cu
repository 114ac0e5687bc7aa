// ts_control.cu -- control-rate stage (S2..S7) and the tick-level phase scan of S9.
//
// One CTA per voice.  Per control tick j (tau_j = j*R/sr, S5) a thread evaluates the six ADSRs in
// closed form (S4), the two LFOs (S6; each with its rate and amp ADSR) and the
// modulation mixer (S7), all in fp64 because the two pitch rows feed the oscillator phase (H1 in
// DESIGN.md).  The two running sums over time are done as block-wide prefix scans of Q0.64
// fixed-point fractions of a cycle (warp __shfl_up_sync + per-warp totals + a carry between chunks of
// blockDim ticks): integer addition mod 2^64 is exact and associative, so the scan order cannot change
// a bit and phase does not drift however long the render is.
//   * LFO phase  q_j  = q_0 + sum_{i<j} f_i/cr                          (exclusive, mod 1; S6, D21)
//   * VCO phase  Phi_j = phi_0 + sum_{i<j} S_i, S_i = sum of the R increments of interval i.
//     Inside an interval pitch is linear in n (S8), so the increments are a geometric sequence and
//     S_i = inc_i * expm1(R a)/expm1(a), a = (P_{i+1}-P_i) ln2 / (12 R)  (closed form; exact sum).
// The audio kernel then needs nothing from other threads: every run of 20 samples starts from the
// table entry of its tick.
#include "ts_common.cuh"

__constant__ ts_range c_nebula[TS_NPARAM];

cudaError_t ts_upload_nebula(const ts_range *host78, cudaStream_t st) {
    return cudaMemcpyToSymbolAsync(c_nebula, host78, sizeof(ts_range) * TS_NPARAM, 0, cudaMemcpyHostToDevice, st);
}

// S3 map(u; lo,hi,c,S).  __dmul_rn/__dadd_rn: one rounding per operation (no FMA contraction), so the
// affine parameters come out bit-identical to a plain IEEE evaluation of the same expression.
__device__ double ts_map(double u, const ts_range &r) {
    if (!(u >= 0.0)) u = 0.0;
    if (u > 1.0) u = 1.0;
    if (!r.symmetric) {
        const double v = (r.curve == 1.0) ? u : pow(u, 1.0 / r.curve);
        return __dadd_rn(r.lo, __dmul_rn(r.hi - r.lo, v));
    }
    const double d = __dadd_rn(__dmul_rn(2.0, u), -1.0);
    const double a = fabs(d);
    const double v = (r.curve == 1.0) ? a : pow(a, 1.0 / r.curve);
    const double s = (d > 0.0) ? 1.0 : ((d < 0.0) ? -1.0 : 0.0);
    return __dadd_rn((r.lo + r.hi) / 2.0, __dmul_rn((r.hi - r.lo) / 2.0, s * v));
}

// S4 ramp(t,s,d)^alpha.  pow(0,a) = 0 and pow(1,a) = 1 exactly for a > 0, so the saturated ends skip pow.
__device__ __forceinline__ double ts_ramp_pow(double t, double s, double d, double alpha) {
    const double x = t - s;
    double r;
    if (x >= d) r = 1.0;
    else if (x <= 0.0) r = 0.0;
    else r = x / d;
    if (alpha > 0.0 && (r == 0.0 || r == 1.0)) return r;
    return pow(r, alpha);
}

// E(t) = ramp(t,0,A)^a * [1 - (1-S) ramp(t,A,Dc)^a] * [1 - ramp(t,D,Rl)^a]
__device__ __forceinline__ double ts_adsr(double t, const double *p, double D) {
    const double A = p[0], Dc = p[1], S = p[2], Rl = p[3], al = p[4];
    const double r = ts_ramp_pow(t, D, Rl, al);
    if (r == 1.0) return 0.0;  // a * (...) * (1 - 1) = 0 exactly
    const double a = ts_ramp_pow(t, 0.0, A, al);
    if (a == 0.0) return 0.0;
    const double d = ts_ramp_pow(t, A, Dc, al);
    return __dmul_rn(__dmul_rn(a, __dadd_rn(1.0, -__dmul_rn(1.0 - S, d))), 1.0 - r);
}

// frac of a double as Q0.64
__device__ __forceinline__ unsigned long long ts_frac_q64(double x) {
    const double f = x - floor(x);  // exact, in [0,1)
    return __double2ull_rz(f * 18446744073709551616.0);
}
__device__ __forceinline__ double ts_q64_to_double(unsigned long long q) {
    return __ull2double_rz(q >> 11) * (1.0 / 9007199254740992.0);  // exact truncation to 53 bits, [0,1)
}

// Block-wide exclusive scan (mod 2^64) of two values per thread, in thread order.  Returns the
// exclusive prefix in (a, b) and the block totals in (ta, tb).  sm: 2*32 words of shared scratch.
__device__ __forceinline__ void ts_block_scan2(unsigned long long &a, unsigned long long &b, unsigned long long &ta,
                                               unsigned long long &tb, unsigned long long *sm) {
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
    if (wid == 0) {
        unsigned long long wa = (lane < nw) ? sm[lane] : 0ull, wb = (lane < nw) ? sm[32 + lane] : 0ull;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long ua = __shfl_up_sync(0xffffffffu, wa, o);
            const unsigned long long ub = __shfl_up_sync(0xffffffffu, wb, o);
            if (lane >= o) { wa += ua; wb += ub; }
        }
        sm[lane] = wa; sm[32 + lane] = wb;  // inclusive warp totals
    }
    __syncthreads();
    const unsigned long long oa = wid ? sm[wid - 1] : 0ull, ob = wid ? sm[32 + wid - 1] : 0ull;
    ta = sm[nw - 1]; tb = sm[32 + nw - 1];
    a = oa + ia - a;
    b = ob + ib - b;
    __syncthreads();  // scratch may be reused
}

// S6 LFO value at phase p in [0,1): normalised blend of the five shapes (D11).
__device__ __forceinline__ double ts_lfo_mix(double p, const double *w) {
    double sh[5];
    sh[0] = sinpi(2.0 * p);
    const double t = p + 0.75;
    sh[1] = 4.0 * fabs((t - floor(t)) - 0.5) - 1.0;
    sh[2] = 2.0 * p - 1.0;
    sh[3] = 1.0 - 2.0 * p;
    sh[4] = (p < 0.5) ? 1.0 : -1.0;
    double num = 0.0, den = 0.0;
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        num = __dadd_rn(num, __dmul_rn(w[i], sh[i]));
        den += w[i];
    }
    return (den == 0.0) ? 0.0 : num / den;
}

struct ts_pitch2 {
    double p1, p2;
};

__global__ void __launch_bounds__(1024)
ts_control_kernel(const ts_voice *__restrict__ params, int sr, long long N, int K, ts_tick *__restrict__ table,
                  ts_vhdr *__restrict__ hdr, float *__restrict__ params_human, double *__restrict__ dbg_ctl,
                  unsigned long long *__restrict__ d_active, int full) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double h[TS_NPARAM + 2];
    __shared__ unsigned long long scan_sm[64];
    __shared__ int s_jsil;
    ts_pitch2 *buf = reinterpret_cast<ts_pitch2 *>(smem_raw);  // [2][T + 1]

    const int v = blockIdx.x, tid = threadIdx.x, T = blockDim.x;
    const ts_voice &rec = params[v];
    ts_tick *tab = table + (size_t)v * K;

    // ---- S2/S3: parameter map ----
    if (tid < TS_NPARAM) {
        const double hv = ts_map((double)rec.u[tid], c_nebula[tid]);
        h[tid] = hv;
        if (params_human) params_human[(size_t)v * TS_NPARAM + tid] = (float)hv;
    }
    __syncthreads();

    const double D = h[1];
    const double cr = (double)sr / (double)TS_R;
    const long long J = (N + TS_R - 1) / TS_R;  // control intervals that hold samples
    // The voice is silent for good once the release of all four audible envelopes is over (their
    // ramp is 1, so E = 0 exactly): adsr1, adsr2, lfo1_amp, lfo2_amp.
    const double rl_max = fmax(fmax(h[2 + 3], h[7 + 3]), fmax(h[12 + 3], h[22 + 3]));
    if (tid == 0) {
        long long j = (long long)floor((D + rl_max) * cr) - 2;
        if (j < 0) j = 0;
        if (j > K - 1) j = K - 1;
        // first tick with (tau - D) >= rl_max, evaluated exactly as S4's ramp does
        while (j < K && !(((double)(j * TS_R) / (double)sr) - D >= rl_max)) ++j;
        while (j > 0 && (((double)((j - 1) * TS_R) / (double)sr) - D >= rl_max)) --j;
        if (full) j = K;  // debug exports: evaluate every tick
        s_jsil = (int)j;  // == K if never silent inside the table
        const long long n_act = (j * TS_R < N) ? j * TS_R : N;
        ts_vhdr hd;
        hd.shape = (float)h[74];
        const double fc = 440.0 * exp2((h[0] + h[71] - 69.0) / 12.0);
        const double k = 12000.0 / (fc * log10(fc));
        hd.tanh_c = (float)(1.5707963267948966 * k * 2.0 * 1.4426950408889634);
        hd.nk0 = rec.noise_key[0];
        hd.nk1 = rec.noise_key[1];
        hd.n_act = (int32_t)n_act;
        hd.n_ticks = (int32_t)((j + 1 < K) ? j + 1 : K);
        hd.pad[0] = hd.pad[1] = 0;
        hdr[v] = hd;
        if (d_active) atomicAdd(d_active, (unsigned long long)n_act);
    }
    __syncthreads();
    const int jsil = s_jsil;
    const int n_ticks = (jsil + 1 < K) ? jsil + 1 : K;

    // mixer gains folded into the amp rows (S13/S14): l_i / (l1+l2+l3); VCO2 also carries (1 - s/2) of S11
    const double lsum = (h[75] + h[76]) + h[77];
    const double g1 = (lsum == 0.0) ? 0.0 : h[75] / lsum;
    const double g2 = (lsum == 0.0) ? 0.0 : h[76] / lsum * (1.0 - h[74] / 2.0);
    const double g3 = (lsum == 0.0) ? 0.0 : h[77] / lsum;
    const double base1 = h[0] + h[68], base2 = h[0] + h[71];
    const double dep1 = h[69], dep2 = h[72];
    const double f0 = 440.0 / (double)sr;

    unsigned long long carry_q1 = ts_frac_q64(h[34]), carry_q2 = ts_frac_q64(h[42]);
    unsigned long long carry_p1 = ts_frac_q64(h[70]), carry_p2 = ts_frac_q64(h[73]);

    const int nch = (n_ticks + T - 1) / T;
    for (int c = 0; c <= nch; ++c) {
        // ================= phase 1: controls at tick j =================
        const int j = c * T + tid;
        const bool live = (c < nch) && (j < n_ticks);
        double E[6] = {0, 0, 0, 0, 0, 0};
        unsigned long long dq1 = 0, dq2 = 0;
        if (live) {
            const double tau = (double)((long long)j * TS_R) / (double)sr;
#pragma unroll
            for (int e = 0; e < 6; ++e) E[e] = ts_adsr(tau, &h[2 + 5 * e], D);
            const double d1 = __dadd_rn(h[32], __dmul_rn(h[33], E[3])) / cr;
            const double d2 = __dadd_rn(h[40], __dmul_rn(h[41], E[5])) / cr;
            dq1 = (unsigned long long)__double2ll_rn((d1 - rint(d1)) * 18446744073709551616.0);
            dq2 = (unsigned long long)__double2ll_rn((d2 - rint(d2)) * 18446744073709551616.0);
        }
        if (c < nch) {
            unsigned long long t1, t2;
            ts_block_scan2(dq1, dq2, t1, t2, scan_sm);
            const unsigned long long q1 = carry_q1 + dq1, q2 = carry_q2 + dq2;
            carry_q1 += t1;
            carry_q2 += t2;
            if (live) {
                const double L1 = __dmul_rn(E[2], ts_lfo_mix(ts_q64_to_double(q1), &h[35]));
                const double L2 = __dmul_rn(E[4], ts_lfo_mix(ts_q64_to_double(q2), &h[43]));
                const double src[4] = {E[0], E[1], L1, L2};
                double M[5];
#pragma unroll
                for (int d = 0; d < 5; ++d) {
                    double num = 0.0, den = 0.0;
#pragma unroll
                    for (int s = 0; s < 4; ++s) {
                        num = __dadd_rn(num, __dmul_rn(h[48 + 4 * d + s], src[s]));
                        den += h[48 + 4 * d + s];
                    }
                    M[d] = (den == 0.0) ? 0.0 : num / den;
                }
                ts_pitch2 pp;
                pp.p1 = __dadd_rn(base1, __dmul_rn(dep1, M[0]));
                pp.p2 = __dadd_rn(base2, __dmul_rn(dep2, M[2]));
                buf[(c & 1) * (T + 1) + tid] = pp;
                float4 a;
                a.x = (float)(M[1] * g1);
                a.y = (float)(M[3] * g2);
                a.z = (float)(M[4] * g3);
                a.w = 0.0f;
                *reinterpret_cast<float4 *>(&tab[j].a1) = a;
                if (dbg_ctl) {
                    double *o = dbg_ctl + (size_t)v * 5 * K;
#pragma unroll
                    for (int d = 0; d < 5; ++d) o[(size_t)d * K + j] = M[d];
                }
            }
        }
        __syncthreads();
        // ================= phase 2: interval jj = (c-1)*T + tid =================
        if (c > 0) {
            const int jj = (c - 1) * T + tid;
            const bool act = (jj + 1 < n_ticks) && (jj < J);
            unsigned long long s1 = 0, s2 = 0;
            double inc1 = 0, inc2 = 0, e1a = 0, e1b = 0, g20a = TS_RUN, g20b = TS_RUN;
            if (act) {
                const ts_pitch2 p0 = buf[((c - 1) & 1) * (T + 1) + tid];
                const ts_pitch2 p1 = (tid + 1 < T) ? buf[((c - 1) & 1) * (T + 1) + tid + 1] : buf[(c & 1) * (T + 1)];
                {
                    inc1 = f0 * exp2((p0.p1 - 69.0) / 12.0);
                    const double a = (p1.p1 - p0.p1) * (0.69314718055994530942 / (12.0 * TS_R));
                    e1a = expm1(a);
                    const double e20 = expm1(TS_RUN * a);
                    const double e40 = e20 * (2.0 + e20), e80 = e40 * (2.0 + e40);
                    const double e100 = e80 + e20 + e80 * e20;
                    g20a = (e1a == 0.0) ? (double)TS_RUN : e20 / e1a;
                    s1 = ts_frac_q64(inc1 * ((e1a == 0.0) ? (double)TS_R : e100 / e1a));
                }
                {
                    inc2 = f0 * exp2((p0.p2 - 69.0) / 12.0);
                    const double a = (p1.p2 - p0.p2) * (0.69314718055994530942 / (12.0 * TS_R));
                    e1b = expm1(a);
                    const double e20 = expm1(TS_RUN * a);
                    const double e40 = e20 * (2.0 + e20), e80 = e40 * (2.0 + e40);
                    const double e100 = e80 + e20 + e80 * e20;
                    g20b = (e1b == 0.0) ? (double)TS_RUN : e20 / e1b;
                    s2 = ts_frac_q64(inc2 * ((e1b == 0.0) ? (double)TS_R : e100 / e1b));
                }
            }
            unsigned long long t1, t2;
            ts_block_scan2(s1, s2, t1, t2, scan_sm);
            const unsigned long long P1 = carry_p1 + s1, P2 = carry_p2 + s2;
            carry_p1 += t1;
            carry_p2 += t2;
            if (act) {
                double4 *dst = reinterpret_cast<double4 *>(&tab[jj]);
                // 16-byte stores (double2) keep the table writes vectorised without 32-byte alignment
                double2 *d2 = reinterpret_cast<double2 *>(dst);
                d2[0] = make_double2(ts_q64_to_double(P1), inc1);
                d2[1] = make_double2(e1a, g20a);
                d2[2] = make_double2(ts_q64_to_double(P2), inc2);
                d2[3] = make_double2(e1b, g20b);
            }
        }
        // buf[(c-1)&1] is rewritten in iteration c+1's phase 1, after the barriers inside this iteration's scan
    }
}

cudaError_t ts_launch_control(const ts_voice *d_params, int B, int sr, int64_t N, int K, ts_tick *table,
                              ts_vhdr *hdr, float *params_human, double *dbg_ctl, unsigned long long *d_active,
                              int full, cudaStream_t st) {
    // few voices: one big CTA per voice (the chip is otherwise idle); many voices: smaller CTAs, several per SM
    const int T = (B <= 296) ? 1024 : 256;
    const size_t smem = 2 * (size_t)(T + 1) * sizeof(ts_pitch2);
    ts_control_kernel<<<B, T, smem, st>>>(d_params, sr, (long long)N, K, table, hdr, params_human, dbg_ctl, d_active, full);
    return cudaGetLastError();
}
