"""Pins for oracle/ (CPU only).  Each test fixes a part of the oracle to something OTHER than the
oracle itself: published known-answer vectors, closed forms, invariants, special cases that reduce
to a textbook routine, or brute force in independent exact / high-precision arithmetic.
Pin numbers P1..P12 and steps S0..S14 refer to SURVEY.md section 8(c); P:Lnnn = PAPER.md line nnn.
"""
import decimal
import json
import math
import os

import numpy as np
import pytest

import oracle as O

HERE = os.path.dirname(os.path.abspath(__file__))
GOLD = os.path.join(HERE, "golden")
SR = 44100


# ----------------------------------------------------------------------------- helpers
def read_kv(path):
    out = {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, v = line.split("=", 1)
        out[k.strip()] = v.strip()
    return out


def fixed_nebula(h):
    """A nebula with lo = hi = h[p]: map() then returns h[p] exactly for any u (S3)."""
    neb = np.zeros(O.NPARAM, dtype=O.NEBULA_DTYPE)
    neb["lo"] = h
    neb["hi"] = h
    neb["curve"] = 1.0
    neb["symmetric"] = 0
    return neb


def neutral_h(D=100.0):
    """Human-unit parameter vector (layout S2) in which everything is switched off/flat:
    all six ADSRs are a constant 1 while t < D (A = Dc = Rl = 0, S = 1, alpha = 1)."""
    h = np.zeros(O.NPARAM)
    h[0], h[1] = 69.0, D
    for e in range(6):
        h[2 + 5 * e: 7 + 5 * e] = [0.0, 0.0, 1.0, 0.0, 1.0]
    for l in range(2):
        h[32 + 8 * l: 40 + 8 * l] = [0.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 0.0]
    return h


def render_h(h, N, sr=SR, noise_key=(1, 2), want_phase=False):
    u = np.full(O.NPARAM, 0.5, dtype=np.float32)
    return O.render_voice(u, np.array(noise_key, dtype=np.uint32), sr, N, fixed_nebula(h), want_phase=want_phase)


def py_philox(ctr, key):
    """Independent re-statement of S0 in Python integers (itself checked against the KATs below)."""
    c = list(ctr); k = list(key)
    for r in range(10):
        if r:
            k[0] = (k[0] + 0x9E3779B9) & 0xFFFFFFFF
            k[1] = (k[1] + 0xBB67AE85) & 0xFFFFFFFF
        p0 = 0xD2511F53 * c[0]; p1 = 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
    return c


def kat_vectors():
    rows = []
    for line in open(os.path.join(GOLD, "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


# ----------------------------------------------------------------------------- P1 Philox
def test_p1_philox_known_answer_vectors():
    rows = kat_vectors()
    assert len(rows) == 3
    for ctr, key, want in rows:
        assert list(O.philox4x32_10(ctr, key)) == want
        assert py_philox(ctr, key) == want


def test_p1_philox_vs_independent_python_random_inputs():
    rng = np.random.default_rng(1)
    for _ in range(200):
        ctr = [int(x) for x in rng.integers(0, 2**32, 4)]
        key = [int(x) for x in rng.integers(0, 2**32, 2)]
        assert list(O.philox4x32_10(ctr, key)) == py_philox(ctr, key)


# ----------------------------------------------------------------------------- P2 sampler layout
def test_p2_sampler_block0_follows_from_kat():
    # seed 0, g 0, block 0 is ctr = 0, key = 0: the first KAT line.  u = (word >> 8) * 2^-24 (S1, D5)
    u, nk = O.sample_params(0, 0, 1)
    want = [(w >> 8) / 2.0**24 for w in kat_vectors()[0][2]]
    assert [float(x) for x in u[0, :4]] == want


def test_p2_sampler_survey_probe_values():
    g = read_kv(os.path.join(GOLD, "survey_probe.txt"))
    u, nk = O.sample_params(0, 0, 1)
    for i in range(4):
        assert float(u[0, i]) == float(g[f"u{i}"])
    b19 = [int(x, 16) for x in g["block19"].split()]
    assert [int(round(float(x) * 2**24)) for x in u[0, 76:78]] == [w >> 8 for w in b19[:2]]
    assert [int(x) for x in nk[0]] == [int(x, 16) for x in g["noise_key"].split()]
    nb = [int(x, 16) for x in g["noise_block0"].split()]
    assert [O.noise_word(nk[0], n) for n in range(4)] == nb
    z = [float(x) for x in g["noise_z0"].split()]
    assert np.allclose([O.noise_value(w) for w in nb], z, atol=5e-9)
    u7, _ = O.sample_params(7, 3, 128)  # g = 3*128 + 5 = 389
    s7 = [int(x, 16) for x in g["seed7_g389_block0"].split()]
    assert [int(round(float(x) * 2**24)) for x in u7[5, :4]] == [w >> 8 for w in s7]


def test_p2_sampler_counter_and_key_layout_64bit():
    # ctr = (block, g lo32, g hi32, stream), key = (seed lo32, seed hi32): exercised with hi parts set
    seed = (0xDEADBEEF << 32) | 0x12345678
    g = (0x3 << 32) | 0x9ABCDEF0
    u, nk = O.sample_params(seed, g, 1)  # batch_index*B + b with B = 1
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for p in range(O.NPARAM):
        w = py_philox([p >> 2, g & 0xFFFFFFFF, g >> 32, 0], key)[p & 3]
        assert float(u[0, p]) == (w >> 8) / 2.0**24
    assert [int(x) for x in nk[0]] == py_philox([0, g & 0xFFFFFFFF, g >> 32, 2], key)[:2]


def test_p2_u_on_24bit_grid_and_uniform():
    u, _ = O.sample_params(0, 0, 512)
    x = u.astype(np.float64) * 2**24
    assert np.all(x == np.round(x)) and x.min() >= 0 and x.max() < 2**24
    # P:L143 "sampled uniformly": mean 1/2, var 1/12 over 512*78 draws (4-sigma bands)
    n = u.size
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / n)
    assert abs(u.var() - 1 / 12) < 4 * math.sqrt(1 / 180 / n)


def test_p3_sampler_b_invariance():
    a, ka = O.sample_params(5, 0, 256)
    b, kb = O.sample_params(5, 1, 128)
    assert np.array_equal(a[128:], b) and np.array_equal(ka[128:], kb)


# ----------------------------------------------------------------------------- P4 map
def test_p4_map_closed_forms():
    assert O.map_param(0.0, -3, 9, 0.37, 0) == -3 and O.map_param(1.0, -3, 9, 0.37, 0) == 9
    assert O.map_param(0.25, -3, 9, 1.0, 0) == 0.0                       # affine
    assert O.map_param(0.5, 0, 2, 0.5, 0) == 0.5                         # 2 * 0.5^2
    assert O.map_param(0.5, -24, 24, 0.2, 1) == 0.0                      # symmetric centre, exact
    assert O.map_param(0.0, -96, 96, 0.2, 1) == -96 and O.map_param(1.0, -96, 96, 0.2, 1) == 96
    assert O.map_param(0.75, -10, 10, 0.5, 1) == pytest.approx(10 * 0.25, abs=1e-15)  # (2u-1)^2 = .25
    assert O.map_param(0.25, -10, 10, 0.5, 1) == pytest.approx(-10 * 0.25, abs=1e-15)
    assert O.map_param(0.75, -10, 10, 1.0, 1) == 5.0
    # clamp (8(b)): out-of-range and NaN behave as the nearest end / 0
    assert O.map_param(-1, 0, 2, 0.5, 0) == 0 and O.map_param(7, 0, 2, 0.5, 0) == 2
    assert O.map_param(float("nan"), 1, 2, 1, 0) == 1


@pytest.mark.parametrize("c", [0.1, 0.25, 0.5, 1.0, 3.0, 10.0])
def test_p4_map_monotone_and_inverse_round_trip(c):
    us = np.linspace(0, 1, 201)
    for sym in (0, 1):
        # lo = 0 (centre 0 when symmetric) so that tiny u^(1/c) is not absorbed by the offset
        lo, hi = (-4.0, 4.0) if sym else (0.0, 8.0)
        hs = np.array([O.map_param(u, lo, hi, c, sym) for u in us])
        assert np.all(np.diff(hs) >= 0)
        for u, h in zip(us, hs):
            if sym:
                d = h / 4.0
                back = (math.copysign(abs(d) ** c, d) + 1) / 2
            else:
                back = (h / 8.0) ** c
            assert back == pytest.approx(u, abs=1e-9)


def test_p4_c_below_one_favours_low_or_centre():
    assert O.map_param(0.5, 0, 1, 0.25, 0) < 0.5 < O.map_param(0.5, 0, 1, 4.0, 0)
    assert abs(O.map_param(0.75, -1, 1, 0.25, 1)) < 0.5 < abs(O.map_param(0.75, -1, 1, 4.0, 1))


def test_s2_default_nebula_matches_baseline_ranges_and_count():
    neb = O.default_nebula()
    assert len(neb) == 78
    rng = lambda i: (neb["lo"][i], neb["hi"][i])
    assert rng(0) == (0, 127) and rng(1) == (0.01, 1.0)                       # BASELINE.json configs[0]
    for e in range(6):
        b = 2 + 5 * e
        assert rng(b) == rng(b + 1) == rng(b + 3) == (0, 2) and rng(b + 2) == (0, 1) and rng(b + 4) == (0.1, 6)
    for l in range(2):
        b = 32 + 8 * l
        assert rng(b) == (0, 20) and rng(b + 1) == (-10, 10) and rng(b + 2) == (-0.5, 0.5)
        assert neb["symmetric"][b + 1] == 1
    for v in range(2):
        b = 68 + 3 * v
        assert rng(b) == (-24, 24) and rng(b + 1) == (-96, 96) and rng(b + 2) == (-0.5, 0.5)
        assert neb["symmetric"][b] == 1 and neb["symmetric"][b + 1] == 1
    for i in list(range(35, 40)) + list(range(43, 68)) + [74, 75, 76, 77]:
        assert rng(i) == (0, 1)
    assert np.all((neb["curve"] >= 0.1) & (neb["curve"] <= 10))               # P:L270 range of curve


# ----------------------------------------------------------------------------- P5 ADSR
def test_p5_adsr_segment_values():
    A, Dc, S, Rl, al, D = .3, .2, .6, .4, 2.5, 1.0
    f = lambda t: O.adsr(t, A, Dc, S, Rl, al, D)
    assert f(0) == 0 and f(A) == 1
    assert f(A + Dc) == pytest.approx(S, abs=1e-15) and f(.8) == pytest.approx(S, abs=1e-15)
    assert f(D) == pytest.approx(S, abs=1e-15)
    assert f(A / 2) == pytest.approx(0.5 ** al, abs=1e-15) == pytest.approx(0.176776695296637, abs=1e-14)
    assert f(D + Rl / 2) == pytest.approx(S * (1 - 0.5 ** al), abs=1e-15) == pytest.approx(0.493933982822018, abs=1e-14)
    assert f(D + Rl + 1e-9) == 0 and f(3.0) == 0
    assert abs(f(D + Rl)) <= 1e-15
    assert f(A + Dc / 2) == pytest.approx(1 - (1 - S) * 0.5 ** al, abs=1e-15)


def test_p5_adsr_degenerate_and_early_note_off():
    assert O.adsr(0, 0, .2, .6, .4, 2.5, 1.0) == 1                          # A = 0: step already 1 at t = 0
    assert O.adsr(0.0, 0, 0, .6, .4, 2.5, 1.0) == pytest.approx(.6)         # A = Dc = 0: sustain at once
    assert O.adsr(1.0, .1, .1, .5, 0, 1.0, 1.0) == 0                        # Rl = 0: off at t = D
    assert O.adsr(.2, .3, .2, .6, .4, 1.0, .1) == pytest.approx((.2 / .3) * (1 - .1 / .4), abs=1e-15)  # = 0.5
    ts = np.linspace(0, 2, 401)
    lin = np.array([O.adsr(t, .5, .5, .5, .5, 1.0, 1.0) for t in ts])        # alpha = 1: piecewise linear
    want = np.where(ts <= .5, ts / .5, np.where(ts <= 1.0, 1 - .5 * (ts - .5) / .5, .5 * (1 - np.clip((ts - 1) / .5, 0, 1))))
    assert np.allclose(lin, want, atol=1e-14)
    rng = np.random.default_rng(0)
    for _ in range(300):
        A, Dc, Rl = rng.uniform(0, 2, 3); S = rng.uniform(); al = rng.uniform(.1, 6); D = rng.uniform(.01, 1)
        v = [O.adsr(t, A, Dc, S, Rl, al, D) for t in rng.uniform(0, 4, 8)]
        assert min(v) >= 0 and max(v) <= 1


# ----------------------------------------------------------------------------- P6 LFO / controls
def test_p6_lfo_shape_table():
    want = {0.0: [0, 0, -1, 1, 1], 0.25: [1, 1, -.5, .5, 1], 0.5: [0, 0, 0, 0, -1], 0.75: [-1, -1, .5, -.5, -1]}
    for p, w in want.items():
        assert np.allclose(O.lfo_shapes(p), w, atol=3e-16)


def test_p6_lfo_constant_rate_closed_form_and_one_hot():
    N = 4 * SR
    cr = SR / 100
    for shape, fn in [(2, lambda p: 2 * p - 1), (3, lambda p: 1 - 2 * p), (4, lambda p: np.where(p < .5, 1.0, -1.0)),
                      (0, lambda p: np.sin(2 * np.pi * p)), (1, lambda p: 4 * np.abs(((p + .75) % 1) - .5) - 1)]:
        h = neutral_h()
        h[32] = 3.7; h[33] = 0.0; h[34] = 0.125
        h[35:40] = 0; h[35 + shape] = 0.8
        h[48 + 4 * 0 + 2] = 1.0   # vco1 pitch row <- lfo1 only
        E, L, M = O.controls(h, SR, N)
        j = np.arange(O.num_ticks(N))
        p = (0.125 + j * 3.7 / cr) % 1.0           # depth = 0  =>  q_j = q_0 + j f / cr  (exclusive sum)
        ok = np.abs(p - 0.5) > 1e-9                 # keep clear of the square's jump
        assert np.allclose(L[0][ok], fn(p)[ok], atol=1e-11)
        assert np.allclose(M[0][ok], fn(p)[ok], atol=1e-11)   # one-hot mod-mixer row passes the source
        assert np.all(M[1:] == 0)                    # rows with zero weights are exactly 0 (S7)


def test_p6_lfo_rate_and_amp_modulation_by_dedicated_adsrs():
    # each LFO has a rate-mod and an amp-mod ADSR.  Rate ADSR = linear attack over 1 s:
    # f(t) = f0 + dep * t  =>  q_j = q0 + sum_{i<j} (f0 + dep*i/cr)/cr  (arithmetic series, exclusive)
    h = neutral_h()
    h[32], h[33], h[34] = 2.0, 5.0, 0.0
    h[35:40] = [0, 0, 1, 0, 0]                      # saw = 2p - 1: reads the phase back directly
    h[2 + 5 * 3: 7 + 5 * 3] = [1.0, 0, 1, 0, 1]     # lfo1_rate ADSR: A = 1 s, alpha = 1
    h[2 + 5 * 2: 7 + 5 * 2] = [0.5, 0, 1, 0, 1]     # lfo1_amp ADSR: A = 0.5 s, alpha = 1
    N = SR
    cr = SR / 100
    E, L, M = O.controls(h, SR, N)
    j = np.arange(O.num_ticks(N))
    assert np.allclose(E[3], np.minimum(j / cr, 1.0), atol=1e-15)
    q = 2.0 * j / cr + 5.0 * (j * (j - 1) / 2) / cr**2
    jj = j[j <= cr]
    amp = np.minimum(jj / cr / 0.5, 1.0)
    assert np.allclose(L[0][jj], amp * (2 * (q[jj] % 1.0) - 1), atol=1e-10)


def test_d21_lfo_phase_30s_against_exact_rational_sum():
    # D21: the LFO running sum is kept mod 1.  With depth = 0 the increment is the constant double
    # delta = fl(f/cr); exact rational arithmetic gives p_j = frac(q0 + j*delta).  Read p back through a
    # pure saw (2p - 1).  Measured: wrapped sum 1.7e-13 worst, unwrapped fp64 sum 5.7e-11 (q ~ 590, ulp 1.1e-13).
    from fractions import Fraction
    sr, N = 48000, 48000 * 30
    cr = sr / 100
    h = neutral_h(D=1000.0)
    h[32], h[33], h[34] = 19.7, 0.0, -0.3125
    h[35:40] = [0, 0, 1, 0, 0]
    E, L, M = O.controls(h, sr, N)
    delta = Fraction(19.7 / cr)
    for j in list(range(0, 14401, 97)) + [14399, 14400]:
        p = (Fraction(-0.3125) + j * delta) % 1
        got = (L[0][j] + 1) / 2
        d = abs(float(Fraction(got) - p))
        assert min(d, 1 - d) < 1e-12, (j, d)


def test_p6_second_lfo_alone_with_its_own_rate_and_amp_adsrs():
    """LFO 2 on its own ("two LFOs ... each LFO module includes two dedicated ADSRs"): block h[40..47], amp
    envelope e = 4 (h[22..26]), rate envelope e = 5 (h[27..31]) per table S2; LFO 1 and its envelopes carry DIFFERENT
    values, so that reading any of LFO 1's slots instead fails.  Rate ADSR = linear attack over 2 s:
    f(t) = f0 + dep t / 2  =>  q_j = q0 + sum_{i<j} (f0 + dep i / (2 cr)) / cr (exclusive).  Reverse saw 1 - 2p reads the
    phase back; mixer source 3 (lfo2) is routed alone into the vco2-pitch row (d = 2)."""
    h = neutral_h()
    h[40], h[41], h[42] = 3.0, -4.0, 0.25           # lfo2: frequency, rate-mod depth, initial phase
    h[43:48] = [0, 0, 0, 0.6, 0]                    # rsaw only
    h[2 + 5 * 5: 7 + 5 * 5] = [2.0, 0, 1, 0, 1]     # lfo2_rate ADSR (e = 5): A = 2 s, alpha = 1
    h[2 + 5 * 4: 7 + 5 * 4] = [0.25, 0, 1, 0, 1]    # lfo2_amp  ADSR (e = 4): A = 0.25 s, alpha = 1
    h[32], h[33], h[34] = 7.0, 9.0, -0.4            # lfo1: everything different
    h[35:40] = [0, 1, 0, 0, 0]
    h[2 + 5 * 3: 7 + 5 * 3] = [0.7, 0, 1, 0, 1]     # lfo1_rate ADSR (e = 3)
    h[2 + 5 * 2: 7 + 5 * 2] = [1.3, 0, 1, 0, 1]     # lfo1_amp  ADSR (e = 2)
    h[48 + 4 * 2 + 3] = 0.37                        # vco2 pitch row <- lfo2 only
    N = SR
    cr = SR / 100
    E, L, M = O.controls(h, SR, N)
    j = np.arange(O.num_ticks(N))
    t = j / cr
    assert np.allclose(E[5], np.minimum(t / 2.0, 1.0), atol=1e-15)
    assert np.allclose(E[4], np.minimum(t / 0.25, 1.0), atol=1e-15)
    q = 0.25 + 3.0 * j / cr - 4.0 * (j * (j - 1) / 2) / (2.0 * cr**2)
    p = q % 1.0
    ok = np.minimum(p, 1 - p) > 1e-9                # keep clear of the saw's jump
    want = np.minimum(t / 0.25, 1.0) * (1 - 2 * p)
    assert np.allclose(L[1][ok], want[ok], atol=1e-10)
    assert np.allclose(M[2][ok], want[ok], atol=1e-10)      # one-hot on source 3: the row IS lfo2
    assert np.all(M[[0, 1, 3, 4]] == 0)
    assert np.max(np.abs(L[0] - L[1])) > 0.5                # and lfo1 really is something else


def test_s7_modmix_every_row_takes_every_source_from_its_own_slot():
    """w[d][s] = h[48 + 4 d + s] (table S2): a one-hot weight passes source s to row d and to no other row, for all 20
    (d, s) -- the four sources are made distinct constants / signals first."""
    base = neutral_h()
    base[2:7] = [0, 0, 0.25, 0, 1]                  # adsr1 == 0.25
    base[7:12] = [0, 0, 0.75, 0, 1]                 # adsr2 == 0.75
    base[32], base[35:40] = 2.0, [0, 0, 1, 0, 0]    # lfo1: 2 Hz saw
    base[40], base[43:48] = 5.0, [0, 0, 0, 0, 1]    # lfo2: 5 Hz square
    N = 4000
    E0, L0, _ = O.controls(base, SR, N)
    src = [E0[0], E0[1], L0[0], L0[1]]
    assert np.allclose(src[0], 0.25) and np.allclose(src[1], 0.75) and np.ptp(src[2]) > 0.1 and set(np.unique(src[3])) <= {-1.0, 1.0}
    for d in range(5):
        for s_ in range(4):
            h = base.copy()
            h[48 + 4 * d + s_] = 0.3
            E, L, M = O.controls(h, SR, N)
            assert np.allclose(M[d], src[s_], atol=1e-15), (d, s_)
            assert np.all(np.delete(M, d, axis=0) == 0), (d, s_)
    h = base.copy()
    h[48 + 4 * 4: 48 + 4 * 5] = [1, 0, 0, 3]        # noise-amp row: adsr1 and lfo2, weights 1 : 3
    E, L, M = O.controls(h, SR, N)
    assert np.allclose(M[4], (0.25 + 3 * src[3]) / 4, atol=1e-15)


def test_s2_default_nebula_value_by_value():
    """All 78 (lo, hi, curve, symmetric) entries of SURVEY.md 8(c) table S2, typed here from the survey's table (not read
    from the oracle): time-like parameters c = 0.5, LFO rate c = 0.25, pitch modulation depth c = 0.2 symmetric, tuning
    and LFO rate-mod depth symmetric, the rest linear."""
    want = {0: (0, 127, 1, 0), 1: (0.01, 1.0, 0.5, 0)}
    for e in range(6):
        b = 2 + 5 * e
        want[b + 0] = want[b + 1] = want[b + 3] = (0, 2, 0.5, 0)
        want[b + 2] = (0, 1, 1, 0)
        want[b + 4] = (0.1, 6, 1, 0)
    for l in range(2):
        b = 32 + 8 * l
        want[b + 0] = (0, 20, 0.25, 0)
        want[b + 1] = (-10, 10, 0.5, 1)
        want[b + 2] = (-0.5, 0.5, 1, 0)
        for i in range(5):
            want[b + 3 + i] = (0, 1, 1, 0)
    for i in range(48, 68):
        want[i] = (0, 1, 1, 0)
    for v in range(2):
        b = 68 + 3 * v
        want[b + 0] = (-24, 24, 1, 1)
        want[b + 1] = (-96, 96, 0.2, 1)
        want[b + 2] = (-0.5, 0.5, 1, 0)
    for i in range(74, 78):
        want[i] = (0, 1, 1, 0)
    assert sorted(want) == list(range(78))
    neb = O.default_nebula()
    for i in range(78):
        got = (neb["lo"][i], neb["hi"][i], neb["curve"][i], int(neb["symmetric"][i]))
        assert got == want[i], (i, got, want[i])
    assert int(neb["symmetric"].sum()) == 6                                   # 33, 41, 68, 69, 71, 72 and no others


def test_s7_modmix_weighted_mean():
    h = neutral_h()
    h[2:7] = [0, 0, 0.25, 0, 1]      # adsr1 == 0.25
    h[7:12] = [0, 0, 0.75, 0, 1]     # adsr2 == 0.75
    h[48 + 4 * 3 + 0] = 1.0; h[48 + 4 * 3 + 1] = 3.0   # vco2 amp row
    E, L, M = O.controls(h, SR, 1000)
    assert np.allclose(M[3], (1 * .25 + 3 * .75) / 4, atol=1e-16)


# ----------------------------------------------------------------------------- P7 upsample
def test_p7_upsample():
    C = np.array([1.0, 3.0, -2.0, 0.5])
    assert [O.upsample(C, 100 * j) for j in range(3)] == [1.0, 3.0, -2.0]
    assert O.upsample(C, 150) == pytest.approx(0.5) and O.upsample(C, 25) == 1.5
    lin = 0.125 * np.arange(5) - 0.25
    assert all(O.upsample(lin, n) == pytest.approx(0.125 * n / 100 - 0.25, abs=1e-16) for n in range(400))


# ----------------------------------------------------------------------------- P8 VCO / phase scan
def sine_only_h(midi=69.0, phase=0.0):
    h = neutral_h()
    h[0] = midi; h[70] = phase
    h[48 + 4 * 1 + 0] = 1.0      # vco1 amp row <- adsr1 == 1
    h[75] = 1.0                  # mixer: vco1 only
    return h


def test_p8_constant_frequency_sine_is_sin_2pi_f_t():
    N = 4410
    a = render_h(sine_only_h(), N)["audio"]
    n = np.arange(N)
    assert np.abs(a - np.sin(2 * np.pi * 440.0 * n / SR)).max() < 1e-12
    a = render_h(sine_only_h(phase=0.25), N)["audio"]         # phases are in cycles (D12)
    assert np.abs(a - np.cos(2 * np.pi * 440.0 * n / SR)).max() < 1e-12
    a = render_h(sine_only_h(midi=81.0), N)["audio"]          # one octave up: A5 = 880 Hz (D13)
    assert np.abs(a - np.sin(2 * np.pi * 880.0 * n / SR)).max() < 1e-12


def test_p8_period_exactly_100_samples_at_441_hz():
    midi = 69 + 12 * math.log2(441 / 440)
    a = render_h(sine_only_h(midi=midi), 20000)["audio"]
    assert np.abs(a[100:] - a[:-100]).max() < 1e-11
    assert np.abs(a[::100]).max() < 1e-11                     # exclusive sum: sample 0 uses phi_0 = 0


def test_p8_dyadic_increment_phase_is_exact():
    # sr = 3520, MIDI 69 => inc = 440/3520 = 1/8 exactly: phi_n = frac(phi_0 + n/8) with no rounding at all
    r = render_h(sine_only_h(phase=0.0625), 64, sr=3520, want_phase=True)
    assert np.array_equal(r["phase1"], (0.0625 + np.arange(64) / 8.0) % 1.0)
    h = sine_only_h(midi=69 + 24); h[68] = -12.0              # tune adds in semitones: net one octave up
    r = render_h(h, 64, sr=3520, want_phase=True)
    assert np.array_equal(r["phase1"], (np.arange(64) / 4.0) % 1.0)


def _swept_h():
    h = sine_only_h(midi=60.0, phase=-0.3)
    h[2:7] = [0.02, 0.01, 0.4, 0.0, 1.7]   # adsr1 moves within the first ticks
    h[69] = 31.0                           # vco1 mod depth (st)
    h[48 + 4 * 0 + 0] = 1.0                # vco1 pitch row <- adsr1
    return h


def test_p8_brute_force_cumulative_sum_high_precision():
    """phi_n = phi_0 + sum_{k<n} (440/sr) 2^((pitch_k - 69)/12), pitch from upsampled control, re-done in
    50-digit decimal arithmetic from the oracle's own tick values (pins S8 + S9 against a dropped term,
    inclusive/exclusive slip, wrong sign or a semitone/octave mix-up)."""
    h = _swept_h()
    sr, N = 8000, 260
    E, L, M = O.controls(h, sr, N)
    r = render_h(h, N, sr=sr, want_phase=True)
    decimal.getcontext().prec = 50
    Dm = decimal.Decimal
    phi = Dm(h[70])
    ln2 = Dm(2).ln()
    for n in range(N):
        assert abs(float(phi % 1) - r["phase1"][n]) < 1e-13 or abs(abs(float(phi % 1) - r["phase1"][n]) - 1) < 1e-13
        j, m = divmod(n, 100)
        ctl = Dm(M[0][j]) + (Dm(M[0][j + 1]) - Dm(M[0][j])) * Dm(m) / Dm(100)
        pitch = Dm(h[0]) + Dm(h[68]) + Dm(h[69]) * ctl
        phi += Dm(440) / Dm(sr) * ((pitch - 69) / 12 * ln2).exp()


def test_p8_interval_sum_has_geometric_closed_form():
    """Inside one control interval pitch is linear in n, so increments are geometric:
    sum = inc_j * expm1(a R)/expm1(a), a = (pi_{j+1} - pi_j) ln2 / (12 R)."""
    h = _swept_h()
    sr, N = 8000, 500
    E, L, M = O.controls(h, sr, N)
    r = render_h(h, N, sr=sr, want_phase=True)
    ph = np.unwrap(2 * np.pi * r["phase1"]) / (2 * np.pi)
    for j in range(4):
        pj = h[0] + h[68] + h[69] * M[0][j]; pj1 = h[0] + h[68] + h[69] * M[0][j + 1]
        inc = 440.0 / sr * 2 ** ((pj - 69) / 12)
        a = (pj1 - pj) * math.log(2) / 1200
        s = inc * (math.expm1(100 * a) / math.expm1(a) if a else 100)
        assert ph[100 * (j + 1)] - ph[100 * j] == pytest.approx(s, rel=1e-13)


def test_p8_long_render_drift_bound_long_double():
    """The oracle wraps phi every step; its own drift over 1.44 M samples at the most extreme pitch is
    checked against an 80-bit long-double accumulation of the same increments (expect << 1e-6 cycles)."""
    h = sine_only_h(midi=127.0)
    h[68] = 24.0
    N, sr = 1_440_000, 48000
    r = render_h(h, N, sr=sr, want_phase=True)
    inc = np.longdouble(440.0) / np.longdouble(sr) * np.exp2((np.longdouble(127.0 + 24.0) - 69) / 12)
    for n in (1, 10**5, 10**6, N - 1):
        want = float((np.longdouble(n) * inc) % 1)
        d = abs(r["phase1"][n] - want)
        assert min(d, 1 - d) < 1e-6


# ----------------------------------------------------------------------------- P9 silence, mixer
def test_p9_exact_silence_after_last_release():
    u, nk = O.sample_params(0, 0, 16)
    N = 4 * SR
    for b in range(16):
        r = O.render_voice(u[b], nk[b], SR, N, want_human=True)
        h = r["human"]
        t_end = h[1] + max(h[5], h[10], h[15], h[25])       # D + max release of adsr1, adsr2, lfo1_amp, lfo2_amp
        n0 = 100 * (math.ceil(t_end * SR / 100) + 1)
        if n0 < N:
            assert np.all(r["audio"][n0:] == 0)
            assert np.any(r["audio"][: n0] != 0)


def test_p9_zero_levels_and_one_hot_mixer():
    h = sine_only_h(); h[75] = 0.0
    assert np.all(render_h(h, 500)["audio"] == 0)               # sum of levels 0 -> 0 (S13-14)
    h = sine_only_h(); h[75] = 0.0; h[77] = 0.3; h[48 + 4 * 4 + 0] = 1.0   # noise only, a3 == 1
    a = render_h(h, 400, noise_key=(7, 9))["audio"]
    z = np.array([O.noise_value(O.noise_word(np.array([7, 9], dtype=np.uint32), n)) for n in range(400)])
    assert np.allclose(a, z, atol=1e-16)                        # P11: noise-only voice = a3(n) z_n
    h = sine_only_h(); h[75] = 0.2; h[76] = 0.6                 # vco2 level on but its amp row is 0
    a = render_h(h, 400)["audio"]
    assert np.allclose(a, 0.25 * np.sin(2 * np.pi * 440 * np.arange(400) / SR), atol=1e-13)


def test_s13_vca_uses_upsampled_amp_row():
    h = sine_only_h()
    h[2:7] = [2000 / SR, 0, 1, 0, 1]                            # adsr1: linear attack ending ON tick 20
    a = render_h(h, 4410)["audio"]
    n = np.arange(4410)
    env = np.minimum(n / 2000, 1.0)                              # piecewise linear with its kink on a tick
                                                                 # => upsampling reproduces it (P7)
    assert np.abs(a - env * np.sin(2 * np.pi * 440 * n / SR)).max() < 1e-12


# ----------------------------------------------------------------------------- P10 squaresaw
def test_p10_squaresaw_properties():
    for k in (0.051, 3.0, 700.0, 18910.0):
        for s in (0.0, 0.37, 1.0):
            th = np.linspace(0.01, 6.27, 97)
            y = np.array([O.squaresaw(t, k, s) for t in th])
            ym = np.array([O.squaresaw(-t, k, s) for t in th])
            assert np.allclose(y, -ym, atol=1e-15)                           # odd in theta
            assert np.abs(y).max() <= 1.125 + 1e-12
    assert O.squaresaw(1.0, 5000.0, 0.0) == pytest.approx(1.0, abs=1e-12)      # s = 0, large k: +-1
    assert O.squaresaw(4.0, 5000.0, 0.0) == pytest.approx(-1.0, abs=1e-12)
    assert O.squaresaw(0.7, 1e-4, 0.0) == pytest.approx(math.pi / 2 * 1e-4 * math.sin(0.7), rel=1e-6)
    assert abs(O.squaresaw(math.pi, 50.0, 1.0)) < 1e-12                       # s = 1: zero at theta = pi
    assert O.squaresaw(math.pi / 2, 1e6, 1.0) == pytest.approx(0.5, abs=1e-12)  # (1 - 1/2) * 1 * (1 + 0)
    assert O.squaresaw(math.pi / 3, 1e6, 1.0) == pytest.approx(0.75, abs=1e-12)  # (1/2)(1 + cos 60deg)


def test_s11_steepness_k_formula_and_range():
    assert O.squaresaw_k(69.0, 0.0) == pytest.approx(12000 / (440 * math.log10(440)), rel=1e-15)
    k_lo = O.squaresaw_k(127.0, 24.0); k_hi = O.squaresaw_k(0.0, -24.0)
    assert k_lo == pytest.approx(0.051, abs=1e-3) and k_hi == pytest.approx(18910, rel=1e-3)


def test_s11_vco2_in_voice_matches_formula():
    h = neutral_h()
    h[0], h[71], h[73], h[74] = 57.0, 3.0, 0.1, 0.6
    h[48 + 4 * 3 + 0] = 1.0; h[76] = 1.0
    N = 2000
    a = render_h(h, N)["audio"]
    fc = 440 * 2 ** ((57 + 3 - 69) / 12)
    k = 12000 / (fc * math.log10(fc))
    th = 2 * np.pi * (0.1 + fc * np.arange(N) / SR)
    want = (1 - 0.3) * np.tanh(np.pi / 2 * k * np.sin(th)) * (1 + 0.6 * np.cos(th))
    assert np.abs(a - want).max() < 1e-9


# ----------------------------------------------------------------------------- P11 noise
def test_p11_noise_moments_and_range():
    key = np.array([0xdd2fc514, 0xadf5a0db], dtype=np.uint32)
    z = np.array([O.noise_value(O.noise_word(key, n)) for n in range(40000)])
    assert z.min() >= -1 and z.max() < 1
    assert abs(z.mean()) < 4 * math.sqrt(1 / 3 / z.size)
    assert abs(z.var() - 1 / 3) < 4 * math.sqrt(4 / 45 / z.size)
    assert abs(np.corrcoef(z[:-1], z[1:])[0, 1]) < 0.03                     # white
    assert O.noise_value(0) == -1.0 and O.noise_value(0xFFFFFFFF) == 1 - 2.0**-23
    # word n is lane n&3 of Philox(key, (n>>2, 0, 0, 1)) (S12)
    assert O.noise_word(key, 4 * 77 + 2) == py_philox([77, 0, 0, 1], [int(key[0]), int(key[1])])[2]


# ----------------------------------------------------------------------------- P12 determinism / causality
def test_p12_prefix_causality_and_determinism():
    u, nk = O.sample_params(0, 0, 3)
    for b in range(3):
        a4 = O.render_voice(u[b], nk[b], SR, 4 * SR)["audio"]
        a1 = O.render_voice(u[b], nk[b], SR, SR)["audio"]
        assert np.array_equal(a1, a4[:SR])
        assert np.array_equal(a1, O.render_voice(u[b], nk[b], SR, SR)["audio"])


def test_d17_num_samples_and_ticks():
    assert O.num_samples(44100, 4.0) == 176400 and O.num_samples(48000, 30) == 1440000   # 4 s
    assert O.num_samples(44100, 0.00001) == 0 and O.num_samples(3, 0.5) == 2
    assert O.num_ticks(176400) == 1765 and O.num_ticks(44100) == 442 and O.num_ticks(101) == 3 and O.num_ticks(1) == 2


def test_p_paper_arithmetic_facts():
    assert round(714e6 / 44100) == 16190                     # 714 MHz <=> ~16200 x real time
    assert round(1e9 * 4 / 3600) == 1111111                  # 1 B x 4 s = 1,111,111 h


# ----------------------------------------------------------------------------- whole voice (unpinned by the paper)
def test_whole_voice_survey_probe_cross_check():
    g = read_kv(os.path.join(GOLD, "survey_probe.txt"))
    u, nk = O.sample_params(0, 0, 1)
    r = O.render_voice(u[0], nk[0], SR, SR, want_human=True)
    a, h = r["audio"], r["human"]
    assert h[0] == pytest.approx(float(g["midi"]), abs=1e-6) and h[1] == pytest.approx(float(g["duration"]), abs=1e-6)
    assert O.squaresaw_k(h[0], h[71]) == pytest.approx(float(g["k"]), abs=1e-6)
    for n in (0, 1, 2, 1000, 22050, 44099):
        assert a[n] == pytest.approx(float(g[f"out{n}"]), abs=1e-8)
    assert math.sqrt(np.mean(a * a)) == pytest.approx(float(g["rms"]), abs=1e-8)
    assert np.abs(a).max() == pytest.approx(float(g["max"]), abs=1e-8)


def test_voice_independence_row_equals_single_render():
    u, nk = O.sample_params(3, 2, 8)
    batch = O.render_batch(u, nk, SR, 3000, threads=4)
    for b in (0, 5, 7):
        assert np.array_equal(batch[b], O.render_voice(u[b], nk[b], SR, 3000)["audio"])


def test_corpus_train_test_split_follows_p_l102():
    """9 * 1024 train, the next 1024 test, etc.; one tenth of the examples are test."""
    assert not any(O.corpus_is_test(g) for g in (0, 1, 1023, 1024, 9 * 1024 - 1))
    assert all(O.corpus_is_test(g) for g in (9 * 1024, 10 * 1024 - 1, 19 * 1024, 20 * 1024 - 1))
    assert not O.corpus_is_test(10 * 1024) and not O.corpus_is_test(18 * 1024 + 1023)
    n = 50 * 10240
    assert sum(O.corpus_is_test(g) for g in range(0, n, 7)) * 7 == pytest.approx(n / 10, rel=1e-3)
    # the same sound is train or test whatever the batch size: whole batches of 128 and of 1024 never straddle
    for B in (128, 1024):
        for batch in (0, 71, 72, 79, 80, 8, 9, 10):
            flags = {O.corpus_is_test(batch * B + b) for b in range(B)}
            assert len(flags) == 1
    assert O.corpus_is_test(72 * 128) and O.corpus_is_test(79 * 128 + 127) and not O.corpus_is_test(80 * 128)
    assert O.corpus_is_test(2**40 * 10240 + 9 * 1024 + 5)        # 64-bit indices


# ----------------------------------------------------------------------------- VCO2 modulated pitch (S9, row M_2, h[71], h[72])
def test_s9_vco2_modulated_phase_brute_force_high_precision():
    """VCO2's phase uses its OWN row (M_2), tuning (h[71]) and depth (h[72]): phi2_n = phi2_0 + sum_{k<n} (440/sr)
    2^((midi + tune_2 + depth_2 up(M_2)(k) - 69)/12), re-done in 50-digit decimal arithmetic from the oracle's own tick
    values.  Row M_2 is one-hot on adsr2 while row M_0 (VCO1) listens to adsr1 with another depth and tuning, so a
    swapped row, tuning or depth index fails; VCO1 is checked in the same render against its own row."""
    h = neutral_h()
    h[0], h[70], h[73] = 58.0, 0.2, -0.35
    h[2:7] = [0.02, 0.01, 0.4, 0.0, 1.7]          # adsr1 moves within the first ticks
    h[7:12] = [0.005, 0.03, 0.2, 0.0, 0.6]        # adsr2 moves differently
    h[68], h[69] = 2.0, 17.0                      # vco1 tuning, depth
    h[71], h[72] = -5.0, -43.0                    # vco2 tuning, depth (negative: pitch falls with the envelope)
    h[48 + 4 * 0 + 0] = 1.0                       # M_0 <- adsr1
    h[48 + 4 * 2 + 1] = 1.0                       # M_2 <- adsr2
    sr, N = 8000, 260
    E, L, M = O.controls(h, sr, N)
    assert np.array_equal(M[0], E[0]) and np.array_equal(M[2], E[1]) and not np.array_equal(E[0], E[1])
    r = render_h(h, N, sr=sr, want_phase=True)
    decimal.getcontext().prec = 50
    Dm = decimal.Decimal
    ln2 = Dm(2).ln()
    for row, tune, depth, start, key in ((0, 68, 69, 70, "phase1"), (2, 71, 72, 73, "phase2")):
        phi = Dm(h[start])
        for n in range(N):
            d = abs(float(phi % 1) - r[key][n])
            assert min(d, 1 - d) < 1e-13, (key, n)
            j, m = divmod(n, 100)
            ctl = Dm(M[row][j]) + (Dm(M[row][j + 1]) - Dm(M[row][j])) * Dm(m) / Dm(100)
            pitch = Dm(h[0]) + Dm(h[tune]) + Dm(h[depth]) * ctl
            phi += Dm(440) / Dm(sr) * ((pitch - 69) / 12 * ln2).exp()


def test_s9_vco2_audio_follows_its_modulated_phase():
    """... and the square/saw is evaluated AT that phase: y2 = orc_squaresaw(2 pi phase2, k(midi, tune_2), s)."""
    h = neutral_h()
    h[0], h[71], h[72], h[73], h[74] = 50.0, 7.0, 30.0, 0.1, 0.3
    h[7:12] = [0.01, 0.02, 0.5, 0.0, 1.3]
    h[48 + 4 * 2 + 1] = 1.0                       # M_2 <- adsr2
    h[48 + 4 * 3 + 0] = 1.0; h[76] = 1.0          # vco2 amp <- adsr1 (constant 1), only vco2 in the mix
    N = 900
    r = render_h(h, N, want_phase=True)
    k = O.squaresaw_k(50.0, 7.0)
    want = np.array([O.squaresaw(2 * np.pi * p, k, 0.3) for p in r["phase2"]])
    assert np.abs(r["audio"] - want).max() < 1e-9
    assert np.abs(np.diff(r["phase2"][:200] % 1)).std() > 0          # the pitch really moves


# ----------------------------------------------------------------------------- tick spacing R as a parameter
def test_r100_functions_reproduce_the_fixed_r_ones_bit_for_bit():
    u, nk = O.sample_params(5, 0, 3)
    for b in range(3):
        h = O.map_all(u[b])
        for a, c in zip(O.controls(h, SR, 4410), O.controls_r(h, SR, 4410, 100)):
            assert np.array_equal(a, c)
        assert np.array_equal(O.render_voice(u[b], nk[b], SR, 2000)["audio"], O.render_voice_r(u[b], nk[b], SR, 2000, 100)["audio"])
    assert O.num_ticks_r(44100, 100) == O.num_ticks(44100) == 442 and O.num_ticks_r(44100, 1) == 44101
    assert O.num_ticks_r(44101, 7) == 6301 + 1


def test_p7_r1_upsampling_is_the_identity():
    """Pin P7: with one tick per sample (R = 1) the interpolation weight m/R is 0 for every n: up(C)(n) == C[n] exactly."""
    rng = np.random.default_rng(3)
    Cs = rng.standard_normal(64)
    for n in range(63):
        assert O.upsample_r(Cs, n, 1) == Cs[n]
    for R in (2, 7, 100):                          # and for any R the tick values are hit and a line is reproduced
        lin = 0.25 + 0.5 * np.arange(10)
        for n in range(9 * R):
            assert O.upsample_r(lin, n, R) == pytest.approx(0.25 + 0.5 * n / R, abs=1e-14)
            if n % R == 0:
                assert O.upsample_r(Cs, n, R) == Cs[n // R]


def test_r1_controls_are_the_closed_forms_at_every_sample():
    """R = 1 (audio-rate control): tick j sits on sample j, tau_j = j/sr.  ADSRs equal orc_adsr(j/sr) (itself pinned by
    P5), and an LFO with no rate modulation has the closed form q_j = q_0 + j f/sr (P6 at cr = sr)."""
    h = neutral_h(D=0.004)
    h[2:7] = [0.001, 0.0015, 0.6, 0.002, 2.5]
    h[32:40] = [250.0, 0.0, 0.125, 1.0, 0.0, 0.0, 0.0, 0.0]     # lfo1: 250 Hz sine, start phase 1/8, no rate modulation
    h[12:17] = [0.0, 0.0, 1.0, 0.0, 1.0]                        # lfo1_amp == 1 while t < D
    h[48 + 4 * 1 + 0] = 1.0                                     # M_1 <- adsr1
    h[48 + 4 * 3 + 2] = 1.0                                     # M_3 <- lfo1
    sr, N = 8000, 80
    E, L, M = O.controls_r(h, sr, N, 1)
    assert E.shape == (6, N + 1)
    for j in range(N + 1):
        t = j / sr
        assert M[1][j] == O.adsr(t, 0.001, 0.0015, 0.6, 0.002, 2.5, 0.004)
        want = math.sin(2 * math.pi * (0.125 + j * 250.0 / sr)) if t < 0.004 else 0.0
        assert M[3][j] == pytest.approx(want, abs=1e-12)
    # the analytic segment values of P5 on the sample grid: E(A) = 1 at j = 8, E(A + Dc) = S at j = 20, 0 after D + Rl
    assert M[1][8] == pytest.approx(1.0, abs=1e-15) and M[1][20] == pytest.approx(0.6, abs=1e-15)
    assert np.all(M[1][49:] == 0.0)


def test_r1_render_constant_sine_and_r_dependence():
    """The audio path with R = 1: a constant-frequency sine is still sin(2 pi f t) (P8), and for a moving envelope
    R = 1 differs from R = 100 exactly as D1 says (the envelope is no longer smeared over 100 samples)."""
    h = sine_only_h()
    u = np.full(O.NPARAM, 0.5, dtype=np.float32)
    nk = np.array([1, 2], dtype=np.uint32)
    a = O.render_voice_r(u, nk, SR, 3000, 1, fixed_nebula(h))["audio"]
    assert np.abs(a - np.sin(2 * np.pi * 440 * np.arange(3000) / SR)).max() < 1e-12
    h[2:7] = [0.003, 0, 1, 0, 1]                                # 132.3-sample linear attack on the amp row
    a1 = O.render_voice_r(u, nk, SR, 400, 1, fixed_nebula(h))["audio"]
    a100 = O.render_voice_r(u, nk, SR, 400, 100, fixed_nebula(h))["audio"]
    n = np.arange(400)
    s = np.sin(2 * np.pi * 440 * n / SR)
    assert np.abs(a1 - np.minimum(n / (0.003 * SR), 1.0) * s).max() < 1e-12          # exact envelope per sample
    e100 = np.interp(n, [0, 100, 200, 300, 400], [0, 100 / 132.3, 1, 1, 1])          # tick values, lerped
    assert np.abs(a100 - e100 * s).max() < 1e-12


# ----------------------------------------------------------------------------- Eq. 2: MMD with the l1 core distance
def test_mmd_identical_sets_is_exactly_zero():
    rng = np.random.default_rng(0)
    X = rng.standard_normal((17, 9))
    v, sums = O.mmd_l1(X, X)
    assert v == 0.0 and sums[0] == sums[1] == sums[2]


def test_mmd_hand_computed_2x2():
    """X = {(0,0), (1,2)}, Y = {(3,0), (0,-1)}.  l1 distances: d(x,y) = [[3,1],[4,4]] -> 12; d(x,x) = [[0,3],[3,0]] -> 6;
    d(y,y) = [[0,4],[4,0]] -> 8.  MMD = (2*12 - 6 - 8) / (2*2) = 2.5   (Eq. 2, 1/n^2 reading)."""
    v, sums = O.mmd_l1(np.array([[0., 0.], [1., 2.]]), np.array([[3., 0.], [0., -1.]]))
    assert list(sums) == [12.0, 6.0, 8.0] and v == 2.5


def test_mmd_invariances_and_scaling():
    rng = np.random.default_rng(1)
    X, Y = rng.standard_normal((23, 11)), rng.standard_normal((23, 11)) + 0.5
    v, sums = O.mmd_l1(X, Y)
    vp, _ = O.mmd_l1(X[rng.permutation(23)], Y[rng.permutation(23)])               # order of the elements
    assert vp == pytest.approx(v, rel=1e-13)
    vs, _ = O.mmd_l1(Y, X)                                                         # symmetric in (X, Y)
    assert vs == pytest.approx(v, rel=1e-13)
    vt, _ = O.mmd_l1(X + 3.25, Y + 3.25)                                           # l1 is translation invariant
    assert vt == pytest.approx(v, rel=1e-12)
    vc, _ = O.mmd_l1(-2.5 * X, -2.5 * Y)                                           # and absolutely homogeneous
    assert vc == pytest.approx(2.5 * v, rel=1e-13)
    assert v > 0                                                                    # shifted sets are apart


def test_mmd_against_an_independent_l1_distance_matrix():
    from scipy.spatial.distance import cdist
    rng = np.random.default_rng(2)
    X, Y = rng.random((40, 32)), rng.random((40, 32)) ** 2
    v, sums = O.mmd_l1(X, Y)
    dxy, dxx, dyy = cdist(X, Y, "cityblock"), cdist(X, X, "cityblock"), cdist(Y, Y, "cityblock")
    assert sums[0] == pytest.approx(dxy.sum(), rel=1e-13) and sums[1] == pytest.approx(dxx.sum(), rel=1e-13)
    assert v == pytest.approx((2 * dxy - dxx - dyy).mean(), rel=1e-12)


def test_16bit_rounding_helpers():
    """round_f16 / round_bf16 (expected values of the 16-bit output formats): round to nearest even on the format's grid."""
    x = np.array([1.0, 1.0 + 2.0 ** -11, 1.0 + 3 * 2.0 ** -11, 0.1, -0.33333, 1.125, 2.0 ** -20])
    assert list(O.round_f16(x)[:3]) == [1.0, 1.0, 1.0 + 2.0 ** -9]                 # ties go to the even code
    assert list(O.round_bf16(np.array([1.0, 1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8]))) == [1.0, 1.0, 1.0 + 2.0 ** -6]
    for f, bits in ((O.round_f16, 11), (O.round_bf16, 8)):
        r = f(x).astype(np.float64)
        assert np.all(np.abs(r - x) <= np.abs(x) * 2.0 ** -bits)                   # within half an ulp
        assert np.array_equal(f(r), r.astype(np.float32))                          # idempotent
