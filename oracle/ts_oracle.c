/*
 * ts_oracle.c -- ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, obviously-correct fp64 CPU implementation of the one hot path of
 * arXiv 2104.12922 ("One Billion Audio Sounds from GPU-enabled Modular Synthesis"):
 * batched rendering of the default modular-synth Voice.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this.  It shares no code, header, table or helper with the CUDA path
 * under paper_2104_12922_b200/csrc/ and include/ .
 *
 * Authority.  PAPER.md (P:Lnnn = /root/reference/PAPER.md line nnn) describes the
 * Voice only at block-diagram level: module census P:L123, two signal rates P:L117,
 * parameter curves P:L143, 78 parameters P:L78, deterministic RNG P:L94.  It prints no
 * DSP equation.  Every formula below is therefore the reading fixed in SURVEY.md
 * section 8(c) (steps S0..S14, readings D1..D20), restated in DESIGN.md "Readings".
 * Each function cites the step it follows.  The arithmetic is written in the order
 * and notation of that section: no blocking, fusion or reordering.
 *
 * Parity status per function (pins live in tests/test_oracle_pins.py):
 *   philox4x32_10 ........ pinned: Random123 known-answer vectors (tests/golden/philox_kat.txt)
 *   sample_params ........ pinned: KAT-derived u[0..3] for (seed 0, g 0); layout by brute force
 *   map_param ............ pinned: closed forms (affine, end points, centre, inverse round trip)
 *   adsr ................. pinned: analytic segment-boundary values
 *   lfo / controls ....... pinned: closed forms with depth 0, one-hot shapes, table of shape values,
 *                          30 s phase against exact rational arithmetic (D21)
 *   upsample ............. pinned: linear signals reproduced, tick values hit
 *   vco phase / sine ..... pinned: sin(2*pi*f*t), exact 100-sample period, exact rational
 *                          cumulative sums on tiny inputs
 *   squaresaw ............ pinned: oddness, limits, zero at theta=pi for s=1, bound 1.125
 *   noise ................ pinned: exact words from the KAT-pinned Philox, moments
 *   controls_r / upsample_r / render_voice_r (tick spacing R as a parameter):
 *                          pinned: R = 1 makes upsampling the identity (P7), per-sample ADSR equals orc_adsr(n/sr),
 *                          LFO closed form at cr = sr, and R = 100 reproduces the fixed-R functions bit for bit
 *   mmd_l1 ............... pinned: MMD(X,X) = 0 exactly, hand-computed 2x2 case, permutation invariance,
 *                          translation invariance, linear scaling, an independent library l1 distance matrix
 *   whole-voice audio .... PARITY UNPINNED by the paper (no printed waveform); cross-checked
 *                          against the survey probe values (last row of pins)
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared -o libts_oracle.so ts_oracle.c -lm
 * (-ffp-contract=off: no fused multiply-add, so every operation rounds once, as written).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_NPARAM 78
#define ORC_R 100 /* control decimation: audio rate / control rate, P:L117 (44.1 kHz / 441 Hz) */

typedef struct {
    double lo, hi, curve;
    int64_t symmetric;
} orc_range;

/* ------------------------------------------------------------------------------------------
 * S0  Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11 -- public algorithm).
 * counter c[4], key k[2], 10 rounds.  Round:
 *   (h0,l0) = mulhilo32(0xD2511F53, c0);  (h1,l1) = mulhilo32(0xCD9E8D57, c2);
 *   c <- (h1^c1^k0, l1, h0^c3^k1, l0);
 * before every round except the first: k0 += 0x9E3779B9, k1 += 0xBB67AE85.
 * ---------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t h0 = (uint32_t)(p0 >> 32), l0 = (uint32_t)p0;
        uint32_t h1 = (uint32_t)(p1 >> 32), l1 = (uint32_t)p1;
        uint32_t n0 = h1 ^ c1 ^ k0;
        uint32_t n1 = l1;
        uint32_t n2 = h0 ^ c3 ^ k1;
        uint32_t n3 = l0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------------------------------
 * S1  sample_params(seed, g).  key = (seed lo32, seed hi32).  Block i = 0..19:
 * ctr = (i, g lo32, g hi32, 0) -> 4 words; parameter p = word (p&3) of block (p>>2).
 * u[p] = (word >> 8) * 2^-24 (exact in fp32, never 1.0; D5).  P:L143 "sampled uniformly
 * from the normalized range"; P:L94 deterministic.  noise_key = first two words of
 * Philox(key, ctr = (0, g lo, g hi, 2)) (D4).
 * ---------------------------------------------------------------------------------------- */
void orc_sample_params(uint64_t seed, uint64_t g, float u[ORC_NPARAM], uint32_t noise_key[2]) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    for (int p = 0; p < ORC_NPARAM; ++p) {
        uint32_t ctr[4] = {(uint32_t)(p >> 2), (uint32_t)g, (uint32_t)(g >> 32), 0u};
        uint32_t w[4];
        orc_philox4x32_10(ctr, key, w);
        u[p] = (float)(w[p & 3] >> 8) * (1.0f / 16777216.0f);
    }
    uint32_t ctr[4] = {0u, (uint32_t)g, (uint32_t)(g >> 32), 2u};
    uint32_t w[4];
    orc_philox4x32_10(ctr, key, w);
    noise_key[0] = w[0];
    noise_key[1] = w[1];
}

/* ------------------------------------------------------------------------------------------
 * S2  Parameter layout and default nebula ("nebula"; values are the survey's
 * PROPOSED table, D6/D8, ranges from BASELINE.json configs[0]).
 * ---------------------------------------------------------------------------------------- */
static void set_range(orc_range *r, double lo, double hi, double curve, int sym) {
    r->lo = lo; r->hi = hi; r->curve = curve; r->symmetric = sym;
}

void orc_default_nebula(orc_range neb[ORC_NPARAM]) {
    set_range(&neb[0], 0.0, 127.0, 1.0, 0);   /* keyboard.midi_f0 */
    set_range(&neb[1], 0.01, 1.0, 0.5, 0);    /* keyboard.duration (s) */
    for (int e = 0; e < 6; ++e) {             /* adsr1, adsr2, lfo1_amp, lfo1_rate, lfo2_amp, lfo2_rate */
        int b = 2 + 5 * e;
        set_range(&neb[b + 0], 0.0, 2.0, 0.5, 0); /* attack (s) */
        set_range(&neb[b + 1], 0.0, 2.0, 0.5, 0); /* decay (s) */
        set_range(&neb[b + 2], 0.0, 1.0, 1.0, 0); /* sustain */
        set_range(&neb[b + 3], 0.0, 2.0, 0.5, 0); /* release (s) */
        set_range(&neb[b + 4], 0.1, 6.0, 1.0, 0); /* alpha */
    }
    for (int l = 0; l < 2; ++l) {
        int b = 32 + 8 * l;
        set_range(&neb[b + 0], 0.0, 20.0, 0.25, 0);  /* lfo.frequency (Hz) */
        set_range(&neb[b + 1], -10.0, 10.0, 0.5, 1); /* lfo.rate_mod_depth (Hz) */
        set_range(&neb[b + 2], -0.5, 0.5, 1.0, 0);   /* lfo.initial_phase (cycles) */
        for (int i = 0; i < 5; ++i) set_range(&neb[b + 3 + i], 0.0, 1.0, 1.0, 0); /* w_sin,tri,saw,rsaw,sqr */
    }
    for (int i = 48; i < 68; ++i) set_range(&neb[i], 0.0, 1.0, 1.0, 0); /* modmix.w[d][s] */
    for (int v = 0; v < 2; ++v) {
        int b = 68 + 3 * v;
        set_range(&neb[b + 0], -24.0, 24.0, 1.0, 1); /* vco.tuning (st) */
        set_range(&neb[b + 1], -96.0, 96.0, 0.2, 1); /* vco.mod_depth (st) */
        set_range(&neb[b + 2], -0.5, 0.5, 1.0, 0);   /* vco.initial_phase (cycles) */
    }
    set_range(&neb[74], 0.0, 1.0, 1.0, 0); /* vco2.shape */
    set_range(&neb[75], 0.0, 1.0, 1.0, 0); /* mixer level vco1 */
    set_range(&neb[76], 0.0, 1.0, 1.0, 0); /* mixer level vco2 */
    set_range(&neb[77], 0.0, 1.0, 1.0, 0); /* mixer level noise */
}

/* ------------------------------------------------------------------------------------------
 * S3  map(u; lo,hi,c,S)  (normalised [0,1] -> human range through a curve, optionally
 * symmetric about the centre; D7: power law u^(1/c)).  u outside [0,1] is clamped (8(b)).
 * ---------------------------------------------------------------------------------------- */
double orc_map(double u, double lo, double hi, double curve, int64_t symmetric) {
    if (!(u >= 0.0)) u = 0.0; /* also catches NaN */
    if (u > 1.0) u = 1.0;
    if (!symmetric) {
        double v = (curve == 1.0) ? u : pow(u, 1.0 / curve);
        return lo + (hi - lo) * v;
    } else {
        double d = 2.0 * u - 1.0;
        double a = fabs(d);
        double v = (curve == 1.0) ? a : pow(a, 1.0 / curve);
        double s = (d > 0.0) ? 1.0 : ((d < 0.0) ? -1.0 : 0.0);
        return (lo + hi) / 2.0 + (hi - lo) / 2.0 * (s * v);
    }
}

void orc_map_all(const float u[ORC_NPARAM], const orc_range neb[ORC_NPARAM], double h[ORC_NPARAM]) {
    for (int p = 0; p < ORC_NPARAM; ++p)
        h[p] = orc_map((double)u[p], neb[p].lo, neb[p].hi, neb[p].curve, neb[p].symmetric);
}

/* ------------------------------------------------------------------------------------------
 * S4  ADSR (D10).  ramp(t,s,d): x = t-s; x >= d -> 1; else x <= 0 -> 0; else x/d
 * (test order matters: d = 0 gives a step that is already 1 at x = 0).
 * E(t) = ramp(t,0,A)^a * [1 - (1-S) ramp(t,A,Dc)^a] * [1 - ramp(t,D,Rl)^a].
 * ---------------------------------------------------------------------------------------- */
static double orc_ramp(double t, double s, double d) {
    double x = t - s;
    if (x >= d) return 1.0;
    if (x <= 0.0) return 0.0;
    return x / d;
}

double orc_adsr(double t, double A, double Dc, double S, double Rl, double alpha, double D) {
    double a = pow(orc_ramp(t, 0.0, A), alpha);
    double d = pow(orc_ramp(t, A, Dc), alpha);
    double r = pow(orc_ramp(t, D, Rl), alpha);
    return a * (1.0 - (1.0 - S) * d) * (1.0 - r);
}

/* number of control ticks, S5: K = ceil(N/R) + 1 (R = ORC_R on the audio path; any R >= 1 for the control-rate
 * functions with a tick-spacing parameter) */
int64_t orc_num_ticks_r(int64_t N, int R) { return (N + R - 1) / R + 1; }
int64_t orc_num_ticks(int64_t N) { return orc_num_ticks_r(N, ORC_R); }

static double orc_frac(double x) { return x - floor(x); }

/* S6 LFO shapes at phase p in [0,1) (D11). */
void orc_lfo_shapes(double p, double sh[5]) {
    const double TWO_PI = 6.283185307179586476925286766559;
    sh[0] = sin(TWO_PI * p);
    sh[1] = 4.0 * fabs(orc_frac(p + 0.75) - 0.5) - 1.0;
    sh[2] = 2.0 * p - 1.0;
    sh[3] = 1.0 - 2.0 * p;
    sh[4] = (p < 0.5) ? 1.0 : -1.0;
}

/* ------------------------------------------------------------------------------------------
 * S5..S7  Control stage: ticks tau_j = j*R/sr, six ADSRs, two LFOs (exclusive phase sum over
 * ticks), modulation mixer.  P:L117 (control rate), P:L123 (each LFO has a rate-mod and an
 * amp-mod ADSR; modulation mixer).
 * Outputs (any may be NULL): E[6][K], L[2][K], M[5][K].
 * ---------------------------------------------------------------------------------------- */
void orc_controls_r(const double h[ORC_NPARAM], int sr, int64_t N, int R, double *E_out, double *L_out, double *M_out) {
    const int64_t K = orc_num_ticks_r(N, R);
    const double cr = (double)sr / (double)R; /* control rate, D2 with R in place of 100 */
    const double D = h[1];
    double q[2] = {h[34], h[42]}; /* q_0 = initial_phase */
    static const int amp_e[2] = {2, 4}, rate_e[2] = {3, 5};
    for (int64_t j = 0; j < K; ++j) {
        double tau = (double)(j * R) / (double)sr;
        double E[6];
        for (int e = 0; e < 6; ++e) {
            const double *a = &h[2 + 5 * e];
            E[e] = orc_adsr(tau, a[0], a[1], a[2], a[3], a[4], D);
            if (E_out) E_out[e * K + j] = E[e];
        }
        double L[2];
        for (int l = 0; l < 2; ++l) {
            const double *lp = &h[32 + 8 * l];
            double f = lp[0] + lp[1] * E[rate_e[l]];
            double p = orc_frac(q[l]);
            double sh[5];
            orc_lfo_shapes(p, sh);
            double num = 0.0, den = 0.0;
            for (int i = 0; i < 5; ++i) {
                num += lp[3 + i] * sh[i];
                den += lp[3 + i];
            }
            double mix = (den == 0.0) ? 0.0 : num / den;
            L[l] = E[amp_e[l]] * mix;
            if (L_out) L_out[l * K + j] = L[l];
            /* exclusive sum: tick j used q_j.  Only frac(q) is ever read, so the running sum is kept
             * mod 1 (reading D21), exactly as S9 does for the VCO phase: the wrap is exact and
             * keeps this oracle's own rounding at ~1e-16 per tick instead of ulp(q) ~ 1e-13 at q ~ 900. */
            q[l] = orc_frac(q[l] + f / cr);
        }
        const double src[4] = {E[0], E[1], L[0], L[1]};
        for (int d = 0; d < 5; ++d) {
            double num = 0.0, den = 0.0;
            for (int s = 0; s < 4; ++s) {
                num += h[48 + 4 * d + s] * src[s];
                den += h[48 + 4 * d + s];
            }
            if (M_out) M_out[d * K + j] = (den == 0.0) ? 0.0 : num / den;
        }
    }
}

void orc_controls(const double h[ORC_NPARAM], int sr, int64_t N, double *E_out, double *L_out, double *M_out) {
    orc_controls_r(h, sr, N, ORC_R, E_out, L_out, M_out);
}

/* S8  Upsample: linear interpolation tick -> sample; tick j sits on sample j*R. */
double orc_upsample_r(const double *C, int64_t n, int R) {
    int64_t j = n / R, m = n % R;
    return C[j] + (C[j + 1] - C[j]) * ((double)m / (double)R);
}
double orc_upsample(const double *C, int64_t n) { return orc_upsample_r(C, n, ORC_R); }

/* S11 SquareSaw waveform value at theta (D14). */
double orc_squaresaw(double theta, double k, double s) {
    const double HALF_PI = 1.5707963267948966192313216916398;
    return (1.0 - s / 2.0) * tanh(HALF_PI * k * sin(theta)) * (1.0 + s * cos(theta));
}

double orc_squaresaw_k(double midi, double tune2) {
    double fc = 440.0 * exp2((midi + tune2 - 69.0) / 12.0);
    return 12000.0 / (fc * log10(fc));
}

/* S12 noise sample n for a voice's noise_key (D5, D15). */
uint32_t orc_noise_word(const uint32_t noise_key[2], uint64_t n) {
    uint32_t ctr[4] = {(uint32_t)(n >> 2), 0u, 0u, 1u};
    uint32_t w[4];
    orc_philox4x32_10(ctr, noise_key, w);
    return w[n & 3];
}

double orc_noise_value(uint32_t x) { return (double)(x >> 8) * (1.0 / 8388608.0) - 1.0; }

/* ------------------------------------------------------------------------------------------
 * S2..S14  Render one voice.  audio[N] (fp64, before the final float rounding); optional
 * phase1[N], phase2[N] (cycles in [0,1)), human[78].  Returns 0, or -1 on allocation failure.
 * ---------------------------------------------------------------------------------------- */
int orc_render_voice_r(const float u[ORC_NPARAM], const uint32_t noise_key[2], const orc_range neb[ORC_NPARAM],
                       int sr, int64_t N, int R, double *audio, double *phase1, double *phase2, double *human) {
    const double TWO_PI = 6.283185307179586476925286766559;
    double h[ORC_NPARAM];
    orc_map_all(u, neb, h);
    if (human) memcpy(human, h, sizeof h);
    const int64_t K = orc_num_ticks_r(N, R);
    double *M = (double *)malloc((size_t)(5 * K) * sizeof(double));
    if (!M) return -1;
    orc_controls_r(h, sr, N, R, NULL, NULL, M);
    const double *M_p1 = M + 0 * K, *M_a1 = M + 1 * K, *M_p2 = M + 2 * K, *M_a2 = M + 3 * K, *M_a3 = M + 4 * K;

    const double midi = h[0];
    const double tune1 = h[68], depth1 = h[69], tune2 = h[71], depth2 = h[72];
    const double shape = h[74];
    const double l1 = h[75], l2 = h[76], l3 = h[77];
    const double lsum = l1 + l2 + l3;
    const double k = orc_squaresaw_k(midi, tune2);
    double phi1 = h[70], phi2 = h[73]; /* phi_0 = initial_phase (cycles) */

    for (int64_t n = 0; n < N; ++n) {
        /* S9: exclusive running sum -- sample n uses phi_n */
        double m1 = orc_upsample_r(M_p1, n, R), m2 = orc_upsample_r(M_p2, n, R);
        double pitch1 = midi + tune1 + depth1 * m1;
        double pitch2 = midi + tune2 + depth2 * m2;
        double inc1 = (440.0 / (double)sr) * exp2((pitch1 - 69.0) / 12.0);
        double inc2 = (440.0 / (double)sr) * exp2((pitch2 - 69.0) / 12.0);
        if (phase1) phase1[n] = orc_frac(phi1);
        if (phase2) phase2[n] = orc_frac(phi2);
        /* S10, S11 */
        double y1 = sin(TWO_PI * phi1);
        double y2 = orc_squaresaw(TWO_PI * phi2, k, shape);
        /* S12 */
        double z = orc_noise_value(orc_noise_word(noise_key, (uint64_t)n));
        /* S13, S14 */
        double a1 = orc_upsample_r(M_a1, n, R), a2 = orc_upsample_r(M_a2, n, R), a3 = orc_upsample_r(M_a3, n, R);
        double out = (lsum == 0.0) ? 0.0 : (l1 * a1 * y1 + l2 * a2 * y2 + l3 * a3 * z) / lsum;
        audio[n] = out;
        phi1 = orc_frac(phi1 + inc1);
        phi2 = orc_frac(phi2 + inc2);
    }
    free(M);
    return 0;
}

int orc_render_voice(const float u[ORC_NPARAM], const uint32_t noise_key[2], const orc_range neb[ORC_NPARAM],
                     int sr, int64_t N, double *audio, double *phase1, double *phase2, double *human) {
    return orc_render_voice_r(u, noise_key, neb, sr, N, ORC_R, audio, phase1, phase2, human);
}

/* D17: N = llround(sr * seconds) */
int64_t orc_num_samples(int sr, double seconds) { return (int64_t)llround((double)sr * seconds); }

/* Train/test designation ("9 * 1024 samples are designated as train, the next 1024 samples as test,
 * etc."; one tenth of the examples).  Global voice index g -> 1 if test. */
int orc_corpus_is_test(uint64_t g) {
    uint64_t block = g / 1024u;      /* blocks of 1024 consecutive sounds */
    return (block % 10u) == 9u;      /* nine train blocks, then one test block */
}

/* ------------------------------------------------------------------------------------------
 * Eq. 2 (Eq. 2 at P:L230): maximum mean discrepancy of two sets X, Y of n elements each with the
 * l1 distance as the core distance d ("OpenL3 ... l1 as the core distance d"):
 *     MMD(X, Y) = 1/(n n) * sum_{i,j} [ 2 d(x_i, y_j) - d(x_i, x_j) - d(y_i, y_j) ].
 * "1/nn" in PAPER.md is garbled; read as 1/n^2 (reading D25), and the sum runs over all n*n ordered pairs
 * (the printed bounds "i,j=0..n" would count n+1 elements of an n-element set).  X, Y: [n][dim] row-major.
 * sums (may be NULL): [0] sum d(x_i,y_j), [1] sum d(x_i,x_j), [2] sum d(y_i,y_j).
 * ---------------------------------------------------------------------------------------- */
double orc_l1(const double *a, const double *b, int dim) {
    double s = 0.0;
    for (int k = 0; k < dim; ++k) s += fabs(a[k] - b[k]);
    return s;
}

double orc_mmd_l1(const double *X, const double *Y, int n, int dim, double sums[3]) {
    double sxy = 0.0, sxx = 0.0, syy = 0.0;
    for (int i = 0; i < n; ++i) {
        for (int j = 0; j < n; ++j) {
            sxy += orc_l1(X + (size_t)i * dim, Y + (size_t)j * dim, dim);
            sxx += orc_l1(X + (size_t)i * dim, X + (size_t)j * dim, dim);
            syy += orc_l1(Y + (size_t)i * dim, Y + (size_t)j * dim, dim);
        }
    }
    if (sums) { sums[0] = sxy; sums[1] = sxx; sums[2] = syy; }
    return (2.0 * sxy - sxx - syy) / ((double)n * (double)n);
}
