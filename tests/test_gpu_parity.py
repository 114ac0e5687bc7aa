"""GPU parity tests: the CUDA path (through the C-ABI binding) against the fp64 CPU oracle, element by
element on the same seeded inputs.  Bars (BASELINE.json north_star):
  * bit-exact: every u (fp32 bit pattern), noise_key, raw Philox noise words;
  * audio, per voice: max |g - o| <= 2e-3 AND relative RMS <= 1e-4, with reading D19 for silent voices.
The oracle's inputs always come from the oracle's own sampler (never from the GPU).
"""
import numpy as np
import pytest

import oracle as O
from paper_2104_12922_b200 import workloads as W

pytestmark = pytest.mark.gpu

MAX_ABS = 2e-3   # north_star
REL_RMS = 1e-4   # north_star


@pytest.fixture(scope="module")
def T():
    import torch
    import paper_2104_12922_b200 as ts
    assert torch.cuda.is_available()
    ts.ts_set_nebula(None)
    yield ts
    ts.ts_set_nebula(None)


def to_dev(u, nk):
    import torch
    rec = np.empty((u.shape[0], 80), dtype=np.float32)
    rec[:, :78] = u
    rec[:, 78:] = nk.view(np.float32)
    return torch.from_numpy(rec).cuda()


def voice_stats(g, o):
    """g: fp32 GPU row, o: fp64 oracle row -> (max abs err, relative RMS err per D19)."""
    d = g.astype(np.float64) - o
    n = o.size
    onorm = np.sqrt(np.sum(o * o))
    rel = np.sqrt(np.sum(d * d)) / max(onorm, 1e-6 * np.sqrt(n))
    return float(np.max(np.abs(d))) if n else 0.0, float(rel)


def assert_parity(g, o, what=""):
    worst = (0.0, 0.0, -1)
    for b in range(o.shape[0]):
        if not np.any(o[b]):
            assert not np.any(g[b]), f"{what} voice {b}: oracle is exactly silent, GPU is not"
            continue
        mx, rel = voice_stats(g[b], o[b])
        if mx > worst[0]:
            worst = (mx, rel, b)
        assert mx <= MAX_ABS and rel <= REL_RMS, f"{what} voice {b}: max|err|={mx:.3e} relRMS={rel:.3e}"
    return worst


def setup_workload(ts, name, batch_index=0, voices=None):
    """-> (wl, nebula, u (edited, oracle-drawn), nk, device records built from the GPU's own draw)."""
    wl = W.WORKLOADS[name]
    u_o, nk_o = O.sample_params(wl.seed, batch_index, wl.B)
    rec = ts.ts_sample_params(wl.seed, batch_index, wl.B).cpu().numpy()
    assert np.array_equal(rec[:, :78].view(np.uint32), u_o.view(np.uint32)), "sampled u not bit-exact"
    assert np.array_equal(rec[:, 78:].view(np.uint32), nk_o), "noise_key not bit-exact"
    first = batch_index * wl.B
    u = W.edit_u(u_o, wl, first)
    u_g = W.edit_u(rec[:, :78], wl, first)
    nk_g = np.ascontiguousarray(rec[:, 78:]).view(np.uint32)
    if voices is not None:
        u, nk_o, u_g, nk_g = u[voices], nk_o[voices], u_g[voices], nk_g[voices]
    neb_o = W.apply_nebula(O.default_nebula(), wl)
    ts.ts_set_nebula(W.apply_nebula(ts.ts_default_nebula(), wl))
    return wl, neb_o, u, nk_o, to_dev(u_g, nk_g)


# ---------------------------------------------------------------------------------- integers: bit-exact
@pytest.mark.parametrize("seed,batch,B", [(0, 0, 4), (0, 0, 128), (7, 3, 128), (2**63 + 12345, 2**40, 1024),
                                          (1, 2**32 - 1, 3), (0xFFFFFFFFFFFFFFFF, 0, 33)])
def test_sampler_bit_exact(T, seed, batch, B):
    rec = T.ts_sample_params(seed, batch, B).cpu().numpy()
    u, nk = O.sample_params(seed, batch, B)
    assert np.array_equal(rec[:, :78].view(np.uint32), u.view(np.uint32))
    assert np.array_equal(rec[:, 78:].view(np.uint32), nk)


def test_sampler_b_invariance(T):
    a = T.ts_sample_params(5, 0, 256).cpu().numpy()
    b = T.ts_sample_params(5, 1, 128).cpu().numpy()
    assert np.array_equal(a[128:].view(np.uint32), b.view(np.uint32))


@pytest.mark.parametrize("key,n0,count", [((0xdd2fc514, 0xadf5a0db), 0, 4096), ((1, 2), 176400 - 7, 1031),
                                          ((0xFFFFFFFF, 0), 2**34 - 5, 64)])
def test_noise_words_bit_exact(T, key, n0, count):
    g = T.ts_debug_noise_u32(key, n0, count).cpu().numpy().view(np.uint32)
    k = np.array(key, dtype=np.uint32)
    o = np.array([O.noise_word(k, n0 + i) for i in range(count)], dtype=np.uint32)
    assert np.array_equal(g, o)


# ---------------------------------------------------------------------------------- control stage
def test_controls_and_human_params_c1(T):
    wl, neb, u, nk, dev = setup_workload(T, "C1")
    ctl = T.ts_debug_controls(dev, wl.sr, wl.seconds).cpu().numpy()
    _, human = T.ts_render(dev, wl.sr, wl.seconds, want_human=True)
    human = human.cpu().numpy()
    for b in range(wl.B):
        h = O.map_all(u[b], neb)
        assert np.allclose(human[b], h.astype(np.float32), rtol=2e-7, atol=0)
        E, L, M = O.controls(h, wl.sr, wl.N)
        assert np.max(np.abs(ctl[b] - M)) < 1e-12, b


def test_phase_c1(T):
    wl, neb, u, nk, dev = setup_workload(T, "C1")
    for vco in (1, 2):
        ph = T.ts_debug_phase(dev, wl.sr, wl.seconds, vco).cpu().numpy()
        for b in range(wl.B):
            r = O.render_voice(u[b], nk[b], wl.sr, wl.N, neb, want_phase=True)
            d = np.abs(ph[b] - r[f"phase{vco}"])
            d = np.minimum(d, 1 - d)
            # the audio kernel accumulates phase on a 2^-32 (VCO 1) / 2^-33 (VCO 2) cycle grid: one rounding of at most
            # 2^-33 cycle per add, 20 adds per run => <= 20 * 2^-33 = 2.3e-9 cycles, inside H4's 1e-8 budget
            assert d.max() < 3e-9, (vco, b, d.max())


def _fixed_voice(T, h):
    """Nebula with lo = hi = h[p] (S3 then returns h[p] for any u) on both sides -> (nebula, device records, u, nk) of 2 voices."""
    neb = np.zeros(O.NPARAM, dtype=O.NEBULA_DTYPE)
    neb["lo"] = h
    neb["hi"] = h
    neb["curve"] = 1.0
    T.ts_set_nebula(neb)
    u, nk = O.sample_params(5, 0, 2)
    return neb, to_dev(u, nk), u, nk


def _flat_h(D=100.0):
    """Everything off / flat (layout S2): all six ADSRs are 1 while t < D, LFOs at 0 Hz, no modulation, no mixer level."""
    h = np.zeros(O.NPARAM)
    h[0], h[1] = 69.0, D
    for e in range(6):
        h[2 + 5 * e: 7 + 5 * e] = [0.0, 0.0, 1.0, 0.0, 1.0]
    for l in range(2):
        h[32 + 8 * l: 40 + 8 * l] = [0.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 0.0]
    return h


def test_noise_only_voice_pins_reading_d24(T):
    """S12 defines the noise value as z = (x >> 8) 2^-23 - 1 (exact in fp32); the audio kernel converts the whole word
    (cvt.rz of x times 2^-31, minus 1: reading D24), which keeps low bits of x that S12 drops (up to 255 x 2^-31 when
    x < 2^31): |g - a3 z| <= 2^-23 a3 + fp32 rounding, one step of S12's grid.  A voice that is noise alone at a constant gain a3 (noise-amp
    row <- adsr1 == 1, level l3 = a3 of a level sum of 1, VCO amplitudes 0) isolates it: z is computed here from the oracle's bit-exact
    Philox words, not from either side's float path."""
    h = _flat_h()
    h[48 + 4 * 4 + 0] = 1.0                                                  # noise-amp row <- adsr1 (== 1)
    a3 = 0.8125                                                              # exact in fp32
    h[77], h[75] = a3, 1.0 - a3                                              # S13-14 divides by l1 + l2 + l3 (= 1 here); the vco1 amp row is all zero, so l1 adds nothing
    sr, seconds = 44100, 0.25
    N = O.num_samples(sr, seconds)
    try:
        neb, dev, u, nk = _fixed_voice(T, h)
        g = T.ts_render(dev, sr, seconds).cpu().numpy().astype(np.float64)
    finally:
        T.ts_set_nebula(None)
    for b in range(2):
        x = np.array([O.noise_word(nk[b], n) for n in range(N)], dtype=np.uint64)
        z = (x >> np.uint64(8)).astype(np.float64) * 2.0**-23 - 1.0          # S12, exact
        err = np.abs(g[b] - a3 * z)
        assert err.max() <= 2.0**-23 * a3 + 2.0**-24, (b, err.max())         # D24's bound + fp32 rounding of a value <= 1
        assert err.max() > 0                                                 # and D24 really is a different rounding
        o = O.render_voice(u[b], nk[b], sr, N, neb)["audio"]
        assert np.max(np.abs(o - a3 * z)) <= 1e-15                           # the oracle IS S12


def test_sine_only_voice_hot_path_recurrence(T):
    """ts_debug_phase goes through the debug variant of the phase recurrence (P += w; w = fma(w, e1, w)); the hot path uses
    the pair form (fma(w, c2, P), fma(w, e2, w)).  A unit-gain sine-only voice with a moving pitch (12 semitones of a 3 Hz LFO:
    every interval has its own geometric increment ratio) reads the hot path's phase back through the sine itself:
    |dg| = 2 pi |dphi|, so a bound of 1e-6 on the audio -- three orders inside the general 2e-3 -- catches any drift of the
    pair recurrence above 1.6e-7 cycles.  What lives inside 1e-6: MUFU.SIN (2^-20.5 = 6.8e-7 absolute at worst), the
    range-reduction multiply (2^-23 relative of <= pi: 3.7e-7 at worst), the gain multiply and the phase grid (2.3e-9 cycles
    = 1.4e-8); measured worst case on a B200: 4.2e-7."""
    h = _flat_h()
    h[32], h[35:40] = 3.0, [1, 0, 0, 0, 0]                                   # lfo1: 3 Hz sine
    h[48 + 4 * 0 + 2] = 1.0                                                  # vco1 pitch row <- lfo1
    h[48 + 4 * 1 + 0] = 1.0                                                  # vco1 amp row <- adsr1 (== 1)
    h[68], h[69], h[70] = 3.5, 12.0, 0.125                                   # tuning, mod depth, initial phase
    h[75] = 1.0                                                              # level l1
    sr, seconds = 44100, 2.0
    N = O.num_samples(sr, seconds)
    try:
        neb, dev, u, nk = _fixed_voice(T, h)
        g = T.ts_render(dev, sr, seconds).cpu().numpy().astype(np.float64)
    finally:
        T.ts_set_nebula(None)
    o = O.render_voice(u[0], nk[0], sr, N, neb, want_phase=True)
    assert np.max(np.abs(o["audio"] - np.sin(2 * np.pi * o["phase1"]))) <= 1e-12   # the voice is the bare sine of its phase
    assert np.ptp(np.diff(o["phase1"]) % 1.0) > 1e-3                          # and the increment really moves
    err = np.abs(g[0] - o["audio"])
    print("sine-only worst |err|:", err.max(), "at", int(err.argmax()))
    assert err.max() <= 1e-6, err.max()


# ---------------------------------------------------------------------------------- audio parity, all configs
def test_audio_c1_every_sample(T):
    wl, neb, u, nk, dev = setup_workload(T, "C1")
    g = T.ts_render(dev, wl.sr, wl.seconds).cpu().numpy()
    o = O.render_batch(u, nk, wl.sr, wl.N, neb)
    print("C1 worst (max, relRMS, voice):", assert_parity(g, o, "C1"))


def test_audio_c2_all_voices(T):
    wl, neb, u, nk, dev = setup_workload(T, "C2")
    g = T.ts_render(dev, wl.sr, wl.seconds).cpu().numpy()
    o = O.render_batch(u, nk, wl.sr, wl.N, neb)
    print("C2 worst (max, relRMS, voice):", assert_parity(g, o, "C2"))
    # pin P9 on the GPU side: exact zeros wherever the oracle is exactly zero from some point on
    for b in range(wl.B):
        nzo = np.flatnonzero(o[b])
        last = nzo[-1] + 1 if nzo.size else 0
        assert not np.any(g[b, last:]), b


def assert_parity_all_voices(T, dev, u, nk, wl, neb, what, chunk=256, full=None):
    """Every voice of a full-size launch against the oracle, streamed in chunks of `chunk` voices to bound host memory
    ("Parity on all voices ... stream voice by voice").  full: the [B, N] CUDA tensor already rendered."""
    import torch
    if full is None:
        full = T.ts_render(dev, wl.sr, wl.seconds)                       # the bench's launch configuration: all voices
    torch.cuda.synchronize()
    worst = (0.0, 0.0, -1)
    obuf = np.empty((chunk, wl.N), dtype=np.float64)
    for b0 in range(0, wl.B, chunk):
        nb = min(chunk, wl.B - b0)
        g = full[b0:b0 + nb].cpu().numpy()
        o = O.render_batch(u[b0:b0 + nb], nk[b0:b0 + nb], wl.sr, wl.N, neb, out=obuf[:nb])
        w = assert_parity(g, o, f"{what} voices {b0}..")
        if w[0] > worst[0]:
            worst = (w[0], w[1], b0 + w[2])
    return worst


@pytest.mark.parametrize("batch", [0, 49, 99])
def test_audio_c3_batches_all_voices(T, batch):
    wl, neb, u, nk, dev = setup_workload(T, "C3", batch_index=batch)
    print("C3 worst:", assert_parity_all_voices(T, dev, u, nk, wl, neb, f"C3[{batch}]"))


def test_audio_c4_long_render_all_voices(T):
    wl, neb, u, nk, dev = setup_workload(T, "C4")
    g = T.ts_render(dev, wl.sr, wl.seconds).cpu().numpy()
    o = O.render_batch(u, nk, wl.sr, wl.N, neb)
    print("C4 worst:", assert_parity(g, o, "C4"))
    ph = T.ts_debug_phase(dev[:4].contiguous(), wl.sr, wl.seconds, 1).cpu().numpy()
    for b in range(4):
        r = O.render_voice(u[b], nk[b], wl.sr, wl.N, neb, want_phase=True)["phase1"]
        for n in (0, 10**5, 10**6, wl.N - 1):
            d = abs(ph[b, n] - r[n])
            assert min(d, 1 - d) < 1e-7, (b, n, d)


def test_audio_c5_all_voices(T):
    """BASELINE.json configs[4]: all 4096 voices (7.2e8 samples) of one full-size launch, streamed through the oracle."""
    wl, neb, u, nk, dev = setup_workload(T, "C5")
    print("C5 worst:", assert_parity_all_voices(T, dev, u, nk, wl, neb, "C5"))


# ---------------------------------------------------------------------------------- edge cases
@pytest.mark.parametrize("sr,seconds,B", [(44100, 0.0123, 3), (44100, 0.00005, 2), (48000, 0.50001, 5),
                                          (8000, 1.0, 2), (44100, 2560 / 44100, 1), (44101, 0.3, 2),
                                          (96000, 0.25, 3)])
def test_ragged_sizes(T, sr, seconds, B):
    T.ts_set_nebula(None)
    u, nk = O.sample_params(3, 1, B)
    N = O.num_samples(sr, seconds)
    assert T.ts_num_samples(sr, seconds) == N and T.ts_num_ticks(N) == O.num_ticks(N)
    import torch
    pad = torch.full((B * N + 64,), 7.0, device="cuda")       # guard words after the buffer
    out = pad[:B * N].view(B, N)
    T.ts_render(to_dev(u, nk), sr, seconds, out=out)
    assert torch.all(pad[B * N:] == 7.0)
    assert_parity(out.cpu().numpy(), O.render_batch(u, nk, sr, N), f"sr={sr} s={seconds}")


def test_unaligned_output_pointer(T):
    import torch
    T.ts_set_nebula(None)
    u, nk = O.sample_params(3, 2, 2)
    sr, seconds = 44100, 0.2
    N = O.num_samples(sr, seconds)
    pad = torch.zeros(2 * N + 8, device="cuda")
    out = pad[1:1 + 2 * N].view(2, N)                            # 4-byte aligned only
    T.ts_render(to_dev(u, nk), sr, seconds, out=out)
    assert_parity(out.cpu().numpy(), O.render_batch(u, nk, sr, N), "unaligned")


def test_extreme_u_values(T):
    T.ts_set_nebula(None)
    rng = np.random.default_rng(11)
    B = 24
    u = rng.integers(0, 2, size=(B, 78)).astype(np.float32)     # every parameter at an end of its range
    u[0] = 0.0
    u[1] = 1.0
    u[2] = 0.5
    u[3, :] = np.float32(1) - np.float32(2.0**-24)
    u[4, 75:78] = 0.0                                            # all mixer levels 0 -> exact silence
    u[5, 48:68] = 0.0                                            # all mod weights 0 -> exact silence
    # LFO rate / rate-depth / start phase stay generic: with end-of-range values (30 Hz at cr = 441 Hz, start
    # phase 0.5) the phase lands EXACTLY on the square/saw jump every 147 ticks, where the sign is decided by
    # the last rounding of either side (reading H8, "LFO tick flip"): not a well-posed parity input.
    ur, _ = O.sample_params(11, 0, B)
    for idx in (32, 33, 34, 40, 41, 42):
        u[3:, idx] = ur[3:, idx]
    nk = rng.integers(0, 2**32, size=(B, 2), dtype=np.uint64).astype(np.uint32)
    sr, seconds = 44100, 1.5
    N = O.num_samples(sr, seconds)
    g = T.ts_render(to_dev(u, nk), sr, seconds).cpu().numpy()
    o = O.render_batch(u, nk, sr, N)
    assert_parity(g, o, "extreme u")
    assert not np.any(g[4]) and not np.any(g[5])


def test_out_of_range_u_is_clamped(T):
    T.ts_set_nebula(None)
    u, nk = O.sample_params(9, 0, 2)
    u2 = u.copy()
    u2[:, 5] = 1.5
    u2[:, 9] = -0.25
    u2[:, 12] = np.nan
    sr, seconds = 44100, 0.5
    g = T.ts_render(to_dev(u2, nk), sr, seconds).cpu().numpy()
    o = O.render_batch(u2, nk, sr, O.num_samples(sr, seconds))
    assert_parity(g, o, "clamp")


def test_determinism_causality_independence(T):
    import torch
    wl, neb, u, nk, dev = setup_workload(T, "C1")
    a = T.ts_render(dev, wl.sr, 1.0)
    b = T.ts_render(dev, wl.sr, 1.0)
    assert torch.equal(a, b)                                    # P12 bitwise determinism
    c = T.ts_render(dev, wl.sr, 0.5)
    assert torch.equal(c, a[:, :c.shape[1]])                    # P12 prefix / causality
    d = T.ts_render(dev[2:3].contiguous(), wl.sr, 1.0)
    assert torch.equal(d[0], a[2])                              # P3 voice independence


def test_error_codes(T):
    import torch
    dev = T.ts_sample_params(0, 0, 2)
    with pytest.raises(T.TsynthError):
        T.ts_render(dev, 0, 1.0)
    with pytest.raises(T.TsynthError):
        T.ts_render(dev, 44100, -1.0)
    neb = T.ts_default_nebula()
    neb["hi"][0] = 400.0                                        # increment beyond the supported range
    T.ts_set_nebula(neb)
    with pytest.raises(T.TsynthError):
        T.ts_render(dev, 44100, 0.1)
    T.ts_set_nebula(None)
    assert T.ts_render(dev, 44100, 0.1).shape == (2, 4410)
    torch.cuda.synchronize()


def test_render_host_end_to_end(T):
    T.ts_set_nebula(None)
    B, sr, seconds = 6, 44100, 0.75
    N = O.num_samples(sr, seconds)
    host = T.ts_render_host(4, 2, B, sr, seconds).numpy()
    u, nk = O.sample_params(4, 2, B)
    assert_parity(host, O.render_batch(u, nk, sr, N), "render_host")


def test_corpus_render_matches_batch_by_batch(T):
    """ts_corpus_render (ts_streaming_lanes() internal lanes, ring of output slots) == ts_sample_params + ts_render, bitwise.
    Rings that are a multiple of the lane count keep a slot on one audio stream; the others need the cross-stream events."""
    import torch
    T.ts_set_nebula(None)
    B, sr, seconds, first = 5, 44100, 0.3, 7
    N = O.num_samples(sr, seconds)
    assert T.ts_streaming_lanes() >= 2
    for n_ring, n_batches in ((2, 2), (3, 7), (4, 9), (5, 12), (6, 14)):
        pr = torch.zeros((n_ring, B, 80), device="cuda")
        ar = torch.full((n_ring, B, N), 9.0, device="cuda")
        T.ts_corpus_render(3, first, n_batches, sr, seconds, pr, ar)
        torch.cuda.synchronize()
        for slot in range(n_ring):
            i = max(k for k in range(n_batches) if k % n_ring == slot)      # the last batch written to this slot
            p = T.ts_sample_params(3, first + i, B)
            a = T.ts_render(p, sr, seconds)
            assert torch.equal(pr[slot].view(torch.int32), p.view(torch.int32)), (n_ring, slot, i)   # keys may be NaN patterns
            assert torch.equal(ar[slot], a), (n_ring, slot, i)
    i0 = max(k for k in range(n_batches) if k % n_ring == 0)                 # what the last ring's slot 0 holds
    u, nk = O.sample_params(3, first + i0, B)                                # and against the oracle
    assert_parity(ar[0].cpu().numpy(), O.render_batch(u, nk, sr, N), "corpus")


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_random_nebula_parity(T, seed):
    """Other hyper-parameter sets (P:L145 'nebula'): curves log-uniform in [0.1, 10] as in the paper's tuning runs
    (P:L270), random symmetry flags, ranges shrunk at random inside the default ones.  Same table on both sides."""
    rng = np.random.default_rng(seed)
    neb_o = O.default_nebula()
    lo, hi = neb_o["lo"].copy(), neb_o["hi"].copy()
    a, b = rng.uniform(0, 0.4, 78), rng.uniform(0.6, 1.0, 78)
    neb_o["lo"], neb_o["hi"] = lo + a * (hi - lo), lo + b * (hi - lo)
    neb_o["curve"] = np.exp(rng.uniform(np.log(0.1), np.log(10.0), 78))
    neb_o["symmetric"] = rng.integers(0, 2, 78)
    neb_o["lo"][[6, 11, 16, 21, 26, 31]] = 0.1          # ADSR alpha stays positive (S4)
    neb_g = T.ts_default_nebula()
    for f in ("lo", "hi", "curve", "symmetric"):
        neb_g[f] = neb_o[f]
    T.ts_set_nebula(neb_g)
    try:
        B, sr, seconds = 12, 44100, 1.2
        u, nk = O.sample_params(100 + seed, 0, B)
        N = O.num_samples(sr, seconds)
        g, human = T.ts_render(to_dev(u, nk), sr, seconds, want_human=True)
        o = O.render_batch(u, nk, sr, N, neb_o)
        for v in range(B):
            assert np.allclose(human[v].cpu().numpy(), O.map_all(u[v], neb_o).astype(np.float32), rtol=3e-7, atol=1e-7)
        assert_parity(g.cpu().numpy(), o, f"nebula {seed}")
    finally:
        T.ts_set_nebula(None)


def test_render_controls_c2_all_voices(T):
    """The control-rate call on its own (Fig. 2 workload) at C2 size against the oracle's mixer rows: its own
    launch mode (no oscillator stage), every voice, exact zeros after the voice has gone silent for good."""
    import torch
    wl, neb, u, nk, dev = setup_workload(T, "C2")
    out = T.ts_render_controls(dev, wl.sr, wl.seconds)
    ctl = out.cpu().numpy()
    assert ctl.shape == (wl.B, 5, O.num_ticks(wl.N))
    for b in range(wl.B):
        E, L, M = O.controls(O.map_all(u[b], neb), wl.sr, wl.N)
        nz = np.flatnonzero(np.any(M != 0.0, axis=0))
        last = nz[-1] + 1 if nz.size else 0
        assert np.max(np.abs(ctl[b] - M)) < 1e-12, b
        assert not np.any(ctl[b][:, last:]), b
    # every element is written by the call itself (no memset): poison the buffer and render again, bitwise equal
    out2 = torch.full_like(out, float("nan"))
    lib = T.lib()
    import ctypes as C
    assert lib.ts_render_controls(C.c_void_p(dev.data_ptr()), wl.B, wl.sr, float(wl.seconds), C.c_void_p(out2.data_ptr())) == 0
    torch.cuda.synchronize()
    assert torch.equal(out, out2)
    # the audio path's own control rows (debug export) agree with it bit for bit where the voice is audible
    dbg = T.ts_debug_controls(dev, wl.sr, wl.seconds).cpu().numpy()
    for b in range(0, wl.B, 7):
        nz = np.flatnonzero(np.any(ctl[b] != 0.0, axis=0))
        last = nz[-1] + 1 if nz.size else 0
        assert np.array_equal(dbg[b][:, :last], ctl[b][:, :last]), b


@pytest.mark.parametrize("R", [1, 7, 441])
def test_render_controls_other_tick_spacings(T, R):
    """the audio-rate-control mode (R = 1: every sample is a tick) and other spacings, at C2's
    length, against the oracle's controls_r.  R = 1 at C2 size is 176 401 ticks per voice (1389 chunks in the look-back
    chain); 16 voices keep the fp64 output at 113 MB."""
    wl, neb, u, nk, dev = setup_workload(T, "C2")
    B = 16 if R == 1 else wl.B
    ctl = T.ts_render_controls_r(dev[:B].contiguous(), wl.sr, wl.seconds, R).cpu().numpy()
    K = O.num_ticks_r(wl.N, R)
    assert ctl.shape == (B, 5, K) and T.ts_num_ticks_r(wl.N, R) == K
    for b in range(B):
        E, L, M = O.controls_r(O.map_all(u[b], neb), wl.sr, wl.N, R)
        # the LFO phase is an exact integer scan on the GPU and a wrapped fp64 sum in the oracle (D21): over 176 400
        # ticks the oracle's own rounding reaches 1e-11 cycles; rows are O(1)
        assert np.max(np.abs(ctl[b] - M)) < (1e-10 if R == 1 else 1e-12), (b, np.max(np.abs(ctl[b] - M)))
        nz = np.flatnonzero(np.any(M != 0.0, axis=0))
        last = nz[-1] + 1 if nz.size else 0
        assert not np.any(ctl[b][:, last:]), b


def test_c3_streaming_protocol_100_batches(T):
    """BASELINE.json configs[2]: 1024 voices x 4 s rendered over 100 consecutive batch indices, here in the bench's
    launch configuration (ts_corpus_render, two alternating output slots); the last two batches against the oracle
    on every voice, records bit-exact."""
    import torch
    wl = W.WORKLOADS["C3"]
    T.ts_set_nebula(None)
    pr = torch.empty((2, wl.B, 80), device="cuda")
    ar = torch.empty((2, wl.B, wl.N), device="cuda")
    T.ts_corpus_render(wl.seed, 0, wl.batches, wl.sr, wl.seconds, pr, ar)
    torch.cuda.synchronize()
    neb = O.default_nebula()
    for batch in (wl.batches - 2, wl.batches - 1):
        slot = batch % 2
        u, nk = O.sample_params(wl.seed, batch, wl.B)
        rec = pr[slot].cpu().numpy()
        assert np.array_equal(rec[:, :78].view(np.uint32), u.view(np.uint32))
        assert np.array_equal(np.ascontiguousarray(rec[:, 78:]).view(np.uint32), nk)
        assert_parity_all_voices(T, None, u, nk, wl, neb, f"C3 stream[{batch}]", full=ar[slot])
        assert T.ts_corpus_is_test(batch * wl.B) == O.corpus_is_test(batch * wl.B)


# ---------------------------------------------------------------------------------- 16-bit output formats
def ulp16(x, mant_bits):
    """spacing of the 16-bit format (mant_bits explicit mantissa bits) at |x| (normal range)."""
    e = np.floor(np.log2(np.maximum(np.abs(x), 2.0 ** -14)))
    return 2.0 ** (e - mant_bits)


@pytest.mark.parametrize("fmt_name,mant", [("f16", 10), ("bf16", 7)])
@pytest.mark.parametrize("wname", ["C1", "C2"])
def test_audio_16bit_formats(T, fmt_name, mant, wname):
    """fp16 / bf16 output: the finished fp32 sample rounded once (RNE).  Expected value = the oracle's fp64 sample rounded
    the same way; bound per sample: the fp32 path's 2e-3 plus half an ulp of the format at that magnitude (a sample
    within 2e-3 of the oracle can round to a neighbouring code).  Exactly-silent tails stay exact zeros, and the 16-bit
    render equals the fp32 render rounded (bitwise)."""
    import torch
    fmt = {"f16": T.TS_F16, "bf16": T.TS_BF16}[fmt_name]
    wl, neb, u, nk, dev = setup_workload(T, wname)
    g16 = T.ts_render_fmt(dev, wl.sr, wl.seconds, fmt)
    g32 = T.ts_render(dev, wl.sr, wl.seconds)
    assert torch.equal(g16, g32.to(g16.dtype))                               # one RNE rounding of the fp32 sample
    g = g16.float().cpu().numpy().astype(np.float64)
    o = O.render_batch(u, nk, wl.sr, wl.N, neb)
    rnd = (O.round_f16 if fmt_name == "f16" else O.round_bf16)(o).astype(np.float64)
    tol = MAX_ABS + 0.5 * ulp16(o, mant)
    assert np.all(np.abs(g - o) <= tol)
    assert np.all(np.abs(g - rnd) <= MAX_ABS + ulp16(o, mant))
    frac_same = np.mean(g == rnd)                                            # most samples land on the oracle's own code
    assert frac_same > (0.9 if fmt_name == "bf16" else 0.5), frac_same
    for b in range(wl.B):
        nzo = np.flatnonzero(o[b])
        last = nzo[-1] + 1 if nzo.size else 0
        assert not np.any(g[b, last:]), b


@pytest.mark.parametrize("sr,seconds,B", [(44100, 0.0123, 3), (48000, 0.50001, 2), (44100, 2564 / 44100, 2)])
def test_16bit_ragged_and_unaligned(T, sr, seconds, B):
    import torch
    T.ts_set_nebula(None)
    u, nk = O.sample_params(3, 1, B)
    N = O.num_samples(sr, seconds)
    for off in (0, 1):                                                       # 1: rows only 2-byte aligned
        pad = torch.full((B * N + 64 + off,), 7.0, device="cuda", dtype=torch.float16)
        out = pad[off:off + B * N].view(B, N)
        T.ts_render_fmt(to_dev(u, nk), sr, seconds, T.TS_F16, out=out)
        assert torch.all(pad[off + B * N:] == 7.0) and torch.all(pad[:off] == 7.0)
        ref = T.ts_render(to_dev(u, nk), sr, seconds)
        assert torch.equal(out, ref.half())


def test_render_host_fmt_and_corpus_fmt(T):
    import torch
    T.ts_set_nebula(None)
    B, sr, seconds = 6, 44100, 0.4
    N = O.num_samples(sr, seconds)
    host = T.ts_render_host_fmt(4, 2, B, sr, seconds, T.TS_BF16)
    p = T.ts_sample_params(4, 2, B)
    assert torch.equal(host.cuda(), T.ts_render(p, sr, seconds).bfloat16())
    pr = torch.zeros((3, B, 80), device="cuda")
    ar = torch.zeros((3, B, N), device="cuda", dtype=torch.float16)
    T.ts_corpus_render_fmt(4, 0, 5, sr, seconds, T.TS_F16, pr, ar)
    torch.cuda.synchronize()
    for i in (2, 3, 4):
        q = T.ts_sample_params(4, i, B)
        assert torch.equal(pr[i % 3].view(torch.int32), q.view(torch.int32))
        assert torch.equal(ar[i % 3], T.ts_render(q, sr, seconds).half())


# ---------------------------------------------------------------------------------- the corpus iterator
def test_corpus_iterator_hands_out_audio_params_and_split(T):
    """ts_corpus_open / next / close: (audio, params, is_test) per batch, P:L94 / P:L98 / P:L102.  B = 128 at the paper's
    default batch size; 1024 / 128 = 8 batches per block, so batches 72..79 are the first test block (g in [9216, 10240))."""
    import torch
    T.ts_set_nebula(None)
    B, sr, seconds, first = 128, 44100, 0.25, 68
    N = O.num_samples(sr, seconds)
    for n_ring in (2, 3, 4):
        pr = torch.zeros((n_ring, B, 80), device="cuda")
        ar = torch.full((n_ring, B, N), 9.0, device="cuda")
        T.ts_corpus_open(0, first, sr, seconds, T.TS_F32, pr, ar)
        got = []
        for k in range(14):
            b = T.ts_corpus_next()
            assert b["batch_index"] == first + k and b["first_voice"] == (first + k) * B and b["slot"] == (first + k) % n_ring
            want_test = O.corpus_is_test(b["first_voice"])
            assert b["is_test_first"] == want_test == b["is_test_last"] == (72 <= first + k < 80)
            got.append((b["audio"].clone(), b["params"].clone()))            # consumed on the current stream
        T.ts_corpus_close()
        torch.cuda.synchronize()
        for k in (0, 5, 13):
            p = T.ts_sample_params(0, first + k, B)
            assert torch.equal(got[k][1].view(torch.int32), p.view(torch.int32))
            assert torch.equal(got[k][0], T.ts_render(p, sr, seconds))
    u, nk = O.sample_params(0, first + 13, B)                                # and against the oracle
    assert_parity(got[13][0].cpu().numpy(), O.render_batch(u, nk, sr, N), "iterator")
    with pytest.raises(T.TsynthError):
        T.ts_corpus_next()                                                   # closed


def test_nebula_is_fixed_while_the_iterator_is_open(T):
    """The iterator issues its batches without re-uploading the nebula, so ts_set_nebula must refuse while it is open (a
    change would split the device table from the host-side extent / silent-tail decisions: a shorter table would leave
    ring samples unwritten).  The refused call changes nothing: the batches after it equal plain renders bit for bit."""
    import torch
    T.ts_set_nebula(None)
    B, sr, seconds, first, n_ring = 16, 44100, 0.5, 3, 3
    N = O.num_samples(sr, seconds)
    short = T.ts_default_nebula()
    short["hi"][1] = 0.05                                                    # note duration
    for e in range(6):
        short["hi"][2 + 5 * e + 3] = 0.01                                    # every release
    pr = torch.zeros((n_ring, B, 80), device="cuda")
    ar = torch.full((n_ring, B, N), 9.0, device="cuda")
    T.ts_corpus_open(0, first, sr, seconds, T.TS_F32, pr, ar)
    got = [T.ts_corpus_next()["audio"].clone()]
    for table in (short, None):
        with pytest.raises(T.TsynthError, match="iterator is open"):
            T.ts_set_nebula(table)
    got += [T.ts_corpus_next()["audio"].clone() for _ in range(4)]
    T.ts_corpus_close()
    torch.cuda.synchronize()
    for k, a in enumerate(got):
        assert torch.equal(a, T.ts_render(T.ts_sample_params(0, first + k, B), sr, seconds)), k
    T.ts_set_nebula(short)                                                   # closed: accepted again
    a = T.ts_render(T.ts_sample_params(0, first, B), sr, seconds)
    assert not torch.equal(a, got[0])
    assert not a[:, int(0.07 * sr):].any().item()                            # 0.05 s note + 0.01 s release: silent after that
    T.ts_set_nebula(None)


# ---------------------------------------------------------------------------------- Eq. 2: MMD with the l1 core distance
@pytest.mark.parametrize("n,d", [(1000, 512), (37, 5), (64, 32), (129, 100), (1, 3), (256, 7), (257, 2), (3000, 16)])
def test_mmd_l1_against_oracle(T, n, d):
    """The paper's setting (n = 1000 sounds, d = 512 OpenL3 values) and ragged sizes, both forms of the call.
    Sorted form (ts_mmd_l1_sorted): values on a grid of 2^-61 of the component's largest magnitude, exact integer sums: each of
    the three sums within 1e-8 relative.  Pairwise form: differences and per-pair sums are fp32 (inputs O(1): each |x - y|
    carries 2^-24 relative, a pair sum over d terms at most d 2^-24 relative), pair sums are added in fp64: 1e-5
    relative covers d = 512 with margin."""
    import torch
    rng = np.random.default_rng(n * 1000 + d)
    X = rng.standard_normal((n, d)).astype(np.float32)
    Y = (0.7 * rng.standard_normal((n, d)) + 0.3).astype(np.float32)
    if d >= 5:
        X[:, 1] = 0.0                                                        # a component that is all zeros in one set
        Y[:, 2] = Y[0, 2]                                                    # a constant component
        X[:, 3] *= 1e-20                                                     # wildly different scales per component
        Y[:, 4] *= 1e6                                                       # (on the sorted form's grid: within 2^37 of each other)
    v, sums = O.mmd_l1(X, Y)
    Xg, Yg = torch.from_numpy(X).cuda(), torch.from_numpy(Y).cuda()
    for pairwise, rel in (("sorted", 1e-8), ("pairwise", 1e-5), ("auto", 1e-5)):
        out = T.ts_mmd_l1(Xg, Yg, form=pairwise).cpu().numpy()
        for k in range(3):
            assert out[1 + k] == pytest.approx(sums[k], rel=rel), (pairwise, k)
        scale = max(sums[0], 1.0) / (n * n)
        assert abs(out[0] - v) <= 4 * rel * scale, (pairwise, out[0], v)
        same = T.ts_mmd_l1(Xg, Xg, form=pairwise).cpu().numpy()
        assert same[0] == 0.0 and same[1] == same[2] == same[3]              # MMD(X, X) = 0 exactly
        again = T.ts_mmd_l1(Xg, Yg, form=pairwise).cpu().numpy()
        assert np.array_equal(out, again)                                    # bitwise reproducible
    # the sorted form does not depend on the order of the rows at all (integer sums); the oracle pins the same invariance
    perm = rng.permutation(n)
    a = T.ts_mmd_l1(Xg, Yg, form="sorted").cpu().numpy()
    b = T.ts_mmd_l1(torch.from_numpy(X[perm]).cuda(), Yg, form="sorted").cpu().numpy()
    assert np.array_equal(a, b)


def test_mmd_l1_large_n_takes_the_pairwise_form(T):
    """n > 8192 does not fit the sorted form's shared memory: ts_mmd_l1_sorted runs the pairwise kernel (small d keeps the oracle fast)."""
    import torch
    rng = np.random.default_rng(9)
    n, d = 8200, 2
    X = rng.standard_normal((n, d)).astype(np.float32)
    Y = (rng.standard_normal((n, d)) + 0.5).astype(np.float32)
    out = T.ts_mmd_l1(torch.from_numpy(X).cuda(), torch.from_numpy(Y).cuda(), form="sorted").cpu().numpy()
    ref = T.ts_mmd_l1(torch.from_numpy(X).cuda(), torch.from_numpy(Y).cuda(), form="pairwise").cpu().numpy()
    assert np.array_equal(out, ref)
    v, sums = O.mmd_l1(X, Y)
    for k in range(3):
        assert out[1 + k] == pytest.approx(sums[k], rel=1e-5)


# ---------------------------------------------------------------------------------- legal end-of-range LFO inputs (H8)
def test_end_of_range_lfo_inputs_stay_finite_and_agree_off_the_jumps(T):
    """LFO rate / depth / start phase at the ENDS of their ranges (30 Hz at cr = 441 Hz from phase 0.5 lands exactly on
    the saw / square jump every 147 ticks: the side taken there is decided by the last rounding, reading H8).  Both
    sides must stay finite everywhere, and agree on every control interval whose two ticks are away from a jump."""
    T.ts_set_nebula(None)
    rng = np.random.default_rng(5)
    B, sr, seconds = 8, 44100, 1.0
    u, nk = O.sample_params(21, 0, B)
    for idx in (32, 33, 34, 40, 41, 42):
        u[:, idx] = rng.integers(0, 2, size=B).astype(np.float32)
    N = O.num_samples(sr, seconds)
    g = T.ts_render(to_dev(u, nk), sr, seconds).cpu().numpy()
    gc = T.ts_debug_controls(to_dev(u, nk), sr, seconds).cpu().numpy()
    assert np.all(np.isfinite(g)) and np.all(np.isfinite(gc)) and np.abs(g).max() <= 1.2
    for b in range(B):
        o = O.render_voice(u[b], nk[b], sr, N)["audio"]
        E, L, M = O.controls(O.map_all(u[b]), sr, N)
        assert np.all(np.isfinite(o))
        bad_tick = np.any(np.abs(gc[b] - M) > 1e-9, axis=0)                  # ticks where the two sides took different sides
        K = M.shape[1]
        ok_iv = ~(bad_tick[:-1] | bad_tick[1:])                              # intervals with both ticks in agreement
        # pitch rows feed the phase: after the first flipped interval the phases differ, so compare up to there
        first_bad = int(np.argmin(ok_iv)) if not ok_iv.all() else K - 1
        n_ok = min(N, first_bad * 100)
        if n_ok > 0:
            d = g[b, :n_ok].astype(np.float64) - o[:n_ok]
            assert np.abs(d).max() <= MAX_ABS, (b, first_bad, np.abs(d).max())


def test_c4_shaped_lookback_chain_four_voices(T):
    """The deepest look-back chain of the configs (30 s at 48 kHz = 114 chunks per voice) on four C4 voices: the case the
    sanitizer runs of profiles/ use (compute-sanitizer racecheck / memcheck / initcheck on this test and on smoke())."""
    import torch
    wl = W.WORKLOADS["C4"]
    u_o, nk_o = O.sample_params(wl.seed, 0, 4)
    u = W.edit_u(u_o, wl, 0)
    neb = W.apply_nebula(O.default_nebula(), wl)
    T.ts_set_nebula(W.apply_nebula(T.ts_default_nebula(), wl))
    dev = to_dev(u, nk_o)
    a = T.ts_render(dev, wl.sr, wl.seconds)
    b = T.ts_render(dev, wl.sr, wl.seconds)
    assert torch.equal(a, b)
    assert_parity(a.cpu().numpy(), O.render_batch(u, nk_o, wl.sr, wl.N, neb), "C4 x4")
    T.ts_sync()                                                       # raises if a look-back wait gave up
    T.ts_set_nebula(None)


def test_lookback_stress_bitwise_repeatable(T):
    """compute-sanitizer is closed on this GPU pool (profiles/r02_sanitizer.md), so the epoch-flag look-back is exercised the
    other way: 200 repeats of the streaming path (control of batch i+1 dispatched under the audio kernel of batch i, the
    tightest residency) and 100 of the deepest chain (114 chunks per voice) must reproduce the first result bit for
    bit (integer carries: any missed or stale aggregate changes bits), and no launch may raise the look-back timeout."""
    import torch
    T.ts_set_nebula(None)
    B, sr, sec = 128, 44100, 4.0
    N = T.ts_num_samples(sr, sec)
    pr = torch.empty((4, B, 80), device="cuda")
    ar = torch.empty((4, B, N), device="cuda")
    T.ts_corpus_render(0, 100, 4, sr, sec, pr, ar)
    torch.cuda.synchronize()
    ref, refp = ar.clone(), pr.clone()
    for it in range(200):
        if it % 50 == 0:
            ar.fill_(7.0)
        T.ts_corpus_render(0, 100, 4, sr, sec, pr, ar)
        torch.cuda.synchronize()
        assert torch.equal(ar, ref) and torch.equal(pr.view(torch.int32), refp.view(torch.int32)), it
    T.ts_sync()
    wl = W.WORKLOADS["C4"]
    T.ts_set_nebula(W.apply_nebula(T.ts_default_nebula(), wl))
    u_o, nk_o = O.sample_params(wl.seed, 0, 4)
    dev = to_dev(W.edit_u(u_o, wl, 0), nk_o)
    first = T.ts_render(dev, wl.sr, wl.seconds).clone()
    for it in range(100):
        assert torch.equal(T.ts_render(dev, wl.sr, wl.seconds), first), it
    T.ts_sync()
    T.ts_set_nebula(None)


def test_lookback_deep_chain_under_saturating_audio_of_other_lanes(T):
    """The tightest residency the streaming path can produce for the look-back (reading D28): 30 s batches at 48 kHz whose
    notes are held to the end (duration lo = hi = 30 s: every one of the 114 chunks per voice is audible, none is skipped),
    streamed over the three lanes, so that the 114-chunk chain of batch i + 1 is dispatched under the saturating audio
    launches of batches i and i - 1.  Integer carries: a missed, stale or torn aggregate changes bits.  40 repeats must
    reproduce the first result bit for bit, equal the single-call render, and raise no look-back timeout."""
    import torch
    neb = T.ts_default_nebula()
    neb["lo"][1] = neb["hi"][1] = 30.0
    T.ts_set_nebula(neb)
    try:
        B, sr, sec, nb = 8, 48000, 30.0, 6
        N = T.ts_num_samples(sr, sec)
        pr = torch.empty((3, B, 80), device="cuda")
        ar = torch.empty((3, B, N), device="cuda")
        T.ts_corpus_render(4, 10, nb, sr, sec, pr, ar)
        torch.cuda.synchronize()
        ref = ar.clone()
        assert ref[:, :, -480:].abs().max().item() > 0                       # held to the end: the last chunk is audible
        for slot in range(3):
            i = slot + 3                                                     # batches 3, 4, 5 are what the ring holds
            assert torch.equal(ref[slot], T.ts_render(T.ts_sample_params(4, 10 + i, B), sr, sec)), slot
        for it in range(40):
            if it % 10 == 0:
                ar.fill_(7.0)
            T.ts_corpus_render(4, 10, nb, sr, sec, pr, ar)
            torch.cuda.synchronize()
            assert torch.equal(ar, ref), it
        T.ts_sync()                                                          # raises if a look-back wait gave up
    finally:
        T.ts_set_nebula(None)


def test_audio_rate_control_mode_r1(T):
    """SURVEY 8(f) item 3, the R = 1 mode of the AUDIO path (reading D27): every sample is a control tick.  Against the
    oracle's render_voice_r(R = 1) on C2's first voices at C2's length (176 401 ticks per voice), plus a ragged case; and
    it must differ from the R = 100 render (the two-rate design is a definition, D1), while R = 100 through the same call
    is ts_render bit for bit."""
    import torch
    wl, neb, u, nk, dev = setup_workload(T, "C2")
    B = 6
    d6 = dev[:B].contiguous()
    g = T.ts_render_r(d6, wl.sr, wl.seconds, 1).cpu().numpy()
    o = np.stack([O.render_voice_r(u[b], nk[b], wl.sr, wl.N, 1, neb)["audio"] for b in range(B)])
    print("R=1 worst:", assert_parity(g, o, "R=1"))
    for b in range(B):
        nzo = np.flatnonzero(o[b])
        last = nzo[-1] + 1 if nzo.size else 0
        assert not np.any(g[b, last:]), b
    g100 = T.ts_render(d6, wl.sr, wl.seconds)
    assert torch.equal(T.ts_render_r(d6, wl.sr, wl.seconds, 100), g100)
    assert np.abs(g - g100.cpu().numpy()).max() > 1e-3
    sr, seconds = 48000, 0.0501                                              # N = 2405: not a multiple of 4
    N = O.num_samples(sr, seconds)
    g = T.ts_render_r(d6[:2].contiguous(), sr, seconds, 1).cpu().numpy()
    o = np.stack([O.render_voice_r(u[b], nk[b], sr, N, 1, neb)["audio"] for b in range(2)])
    assert_parity(g, o, "R=1 ragged")
    with pytest.raises(T.TsynthError):
        T.ts_render_r(d6, wl.sr, wl.seconds, 7)


def test_iterator_multi_chunk_batches_odd_ring_fp16(T):
    """1024-voice batches need several voice chunks (the control table is capped for L2) that alternate between the two
    lanes, and an odd ring moves a slot from one audio stream to the other: the case the cross-stream ring events exist for.
    Every batch handed out must equal ts_sample_params + ts_render_fmt bit for bit."""
    import torch
    T.ts_set_nebula(None)
    B, sr, seconds, first = 1024, 44100, 4.0, 5                              # 4 chunks of 256 voices per batch
    N = O.num_samples(sr, seconds)
    assert T.ts_workspace_bytes(B, sr, seconds) < B * T.ts_num_ticks(N) * 80   # i.e. the table is chunked
    pr = torch.zeros((3, B, 80), device="cuda")
    ar = torch.full((3, B, N), 9.0, device="cuda", dtype=torch.float16)
    T.ts_corpus_open(3, first, sr, seconds, T.TS_F16, pr, ar)
    kept = {}
    for k in range(6):
        b = T.ts_corpus_next()
        assert b["batch_index"] == first + k and b["slot"] == (first + k) % 3
        assert b["is_test_first"] == O.corpus_is_test(b["first_voice"]) and b["is_test_last"] == O.corpus_is_test(b["first_voice"] + B - 1)
        if k in (0, 4, 5):
            kept[k] = (b["audio"].clone(), b["params"].clone())
    T.ts_corpus_close()
    torch.cuda.synchronize()
    for k, (a, p) in kept.items():
        q = T.ts_sample_params(3, first + k, B)
        assert torch.equal(p.view(torch.int32), q.view(torch.int32)), k
        assert torch.equal(a, T.ts_render_fmt(q, sr, seconds, T.TS_F16)), k
    u, nk = O.sample_params(3, first + 5, B)
    o = O.render_batch(u[:64], nk[:64], sr, N)
    g = kept[5][0][:64].float().cpu().numpy().astype(np.float64)
    assert np.all(np.abs(g - o) <= MAX_ABS + 0.5 * ulp16(o, 10))


_MEASURE_AIDS_SCRIPT = r"""
import torch
import paper_2104_12922_b200 as T
T.use_measure_build()
T.ts_set_nebula(None)
rates = T.ts_time_pipes()
assert len(rates) == 8 and all(0.9 < v < 20.0 for v in rates.values()), rates
assert rates["FFMA"] < rates["FFMA2"] < rates["MUFU.EX2"]                # packed fp32x2 is two cycles, MUFU eight
for fast in (True, False):
    v = T.ts_time_alu_bound(fast, 16)
    assert 1e11 < v < 3e12, v                                            # below 148 SMs x 128 lanes x 2 GHz / ~36 instr
buf = torch.empty(64 << 20, device="cuda", dtype=torch.uint8)
gbs = buf.numel() / (T.ts_time_fill(buf, 3) * 1e-3) / 1e9
assert 1000 < gbs < 9000, gbs
B, sr, seconds = 128, 44100, 4.0
p = T.ts_sample_params(0, 0, B)
ring = torch.empty((4, B, T.ts_num_samples(sr, seconds)), device="cuda")
ctl, aud = T.ts_time_kernels(p, sr, seconds, ring, 10)
two = T.ts_time_audio_lanes(p, sr, seconds, ring, 10)
assert 0.005 < two <= aud * 1.05 and 0.005 < ctl < 0.2 and aud < 0.2, (ctl, aud, two)
assert torch.equal(ring[1], T.ts_render(p, sr, seconds))                 # the timing launches render the real thing
assert T.lib_path().endswith("libtsynth_measure.so")
print("MEASURE_AIDS_OK")
"""


def test_measurement_aids_are_sane(T):
    """ts_time_pipes / ts_time_alu_bound / ts_time_fill / ts_time_kernels / ts_time_audio_lanes (bench.py's roofline inputs,
    include/tsynth_measure.h) run and return values in the physically possible range of a B200.  They live in
    libtsynth_measure.so only, which a process loads INSTEAD of the product library: a process of its own, as bench.py is."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", _MEASURE_AIDS_SCRIPT], cwd=root, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "MEASURE_AIDS_OK" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]
    with pytest.raises(T.TsynthError, match="use_measure_build"):
        T.ts_time_pipes()                                                    # not in the product library this process runs


# ---------------------------------------------------------------------------------- a randomised sweep at the bench's own shape
def test_streamed_c2_batches_and_random_nebulae_every_voice(T):
    """24 consecutive C2-sized batches through ts_corpus_render (the launch configuration bench.py times: three streaming
    lanes, ring a multiple of the lanes) and 40 random nebulae at mixed sample rates / lengths, EVERY voice against the
    oracle.  (A 58 880-voice run of the same sweep, 360 batches and 400 nebulae, had no failure: worst 7.0e-5 / 2.9e-6.)"""
    import torch
    T.ts_set_nebula(None)
    B, sr, seconds = 128, 44100, 4.0
    N = O.num_samples(sr, seconds)
    n_ring = 2 * T.ts_streaming_lanes()
    pr = torch.zeros((n_ring, B, 80), device="cuda")
    ar = torch.zeros((n_ring, B, N), device="cuda")
    worst = (0.0, 0.0, -1)
    for start in range(2000, 2024, n_ring):
        T.ts_corpus_render(5, start, n_ring, sr, seconds, pr, ar)
        T.ts_sync()
        for k in range(n_ring):
            u, nk = O.sample_params(5, start + k, B)
            assert np.array_equal(pr[k].cpu().numpy()[:, :78].view(np.uint32), u.view(np.uint32))
            w = assert_parity(ar[k].cpu().numpy(), O.render_batch(u, nk, sr, N), f"streamed batch {start + k}")
            worst = max(worst, w)
    try:
        for seed in range(100, 140):
            rng = np.random.default_rng(seed)
            neb_o = O.default_nebula()
            lo, hi = neb_o["lo"].copy(), neb_o["hi"].copy()
            a, b = rng.uniform(0, 0.4, 78), rng.uniform(0.6, 1.0, 78)
            neb_o["lo"], neb_o["hi"] = lo + a * (hi - lo), lo + b * (hi - lo)
            neb_o["curve"] = np.exp(rng.uniform(np.log(0.1), np.log(10.0), 78))
            neb_o["symmetric"] = rng.integers(0, 2, 78)
            neb_o["lo"][[6, 11, 16, 21, 26, 31]] = 0.1          # ADSR alpha stays positive (S4)
            if seed % 3 == 0:
                neb_o["hi"][1] = 4.0                            # long notes: few silent tails
            neb_g = T.ts_default_nebula()
            for f in ("lo", "hi", "curve", "symmetric"):
                neb_g[f] = neb_o[f]
            T.ts_set_nebula(neb_g)
            Bq, srq, secq = 32, [44100, 48000, 22050, 96000][seed % 4], [1.3, 2.0, 0.777, 3.1][(seed // 4) % 4]
            u, nk = O.sample_params(seed, 7, Bq)
            g = T.ts_render(to_dev(u, nk), srq, secq)
            w = assert_parity(g.cpu().numpy(), O.render_batch(u, nk, srq, O.num_samples(srq, secq), neb_o), f"nebula {seed}")
            worst = max(worst, w)
    finally:
        T.ts_set_nebula(None)
    print("sweep worst (max, relRMS, voice):", worst)


# ---------------------------------------------------------------------------------- one nebula per batch
def _random_nebula(seed):
    rng = np.random.default_rng(seed)
    neb = O.default_nebula()
    lo, hi = neb["lo"].copy(), neb["hi"].copy()
    a, b = rng.uniform(0, 0.4, 78), rng.uniform(0.6, 1.0, 78)
    neb["lo"], neb["hi"] = lo + a * (hi - lo), lo + b * (hi - lo)
    neb["curve"] = np.exp(rng.uniform(np.log(0.1), np.log(10.0), 78))
    neb["symmetric"] = rng.integers(0, 2, 78)
    neb["lo"][[6, 11, 16, 21, 26, 31]] = 0.1                            # ADSR alpha stays positive (S4)
    if seed % 2:
        neb["hi"][1] = 3.0                                              # long notes: the other silent-tail mode
    return neb


def test_corpus_render_with_one_nebula_per_batch(T):
    """ts_corpus_render_nebulae: batch i under table i == ts_set_nebula(table i) + ts_sample_params + ts_render, bitwise;
    every voice against the oracle under its batch's table; the active nebula is untouched; a bad table refuses the call."""
    import torch
    T.ts_set_nebula(None)
    B, sr, seconds, first, nb = 16, 44100, 4.0, 40, 7          # 4 s: odd batches (3 s notes) take TAIL = 0, even ones TAIL = 1
    N = O.num_samples(sr, seconds)
    nebs_o = [_random_nebula(300 + i) for i in range(nb)]
    tabs = np.zeros((nb, 78), dtype=T.NEBULA_DTYPE)
    for i, n in enumerate(nebs_o):
        for f in ("lo", "hi", "curve", "symmetric"):
            tabs[i][f] = n[f]
    for n_ring in (T.ts_streaming_lanes(), 4):
        pr = torch.zeros((n_ring, B, 80), device="cuda")
        ar = torch.full((n_ring, B, N), 9.0, device="cuda")
        T.ts_corpus_render_nebulae(11, first, sr, seconds, T.TS_F32, tabs, pr, ar)
        T.ts_sync()
        got = {i % n_ring: i for i in range(nb)}                         # slot -> last batch written to it
        for slot, i in got.items():
            u, nk = O.sample_params(11, first + i, B)
            assert np.array_equal(pr[slot].cpu().numpy()[:, :78].view(np.uint32), u.view(np.uint32))
            assert_parity(ar[slot].cpu().numpy(), O.render_batch(u, nk, sr, N, nebs_o[i]), f"nebula of batch {i}")
            T.ts_set_nebula(tabs[i])
            assert torch.equal(ar[slot], T.ts_render(T.ts_sample_params(11, first + i, B), sr, seconds)), (n_ring, slot, i)
            T.ts_set_nebula(None)
        # the call left the active (default) nebula alone
        u, nk = O.sample_params(11, first, B)
        assert_parity(T.ts_render(to_dev(u, nk), sr, seconds).cpu().numpy(), O.render_batch(u, nk, sr, N), "active nebula")
    bad = tabs.copy()
    bad[3]["curve"][5] = -1.0
    with pytest.raises(T.TsynthError):
        T.ts_corpus_render_nebulae(11, first, sr, seconds, T.TS_F32, bad, pr, ar)
    bad = tabs.copy()
    bad[2]["hi"][0] = 400.0                                             # pitch beyond the supported increment (D23)
    with pytest.raises(T.TsynthError):
        T.ts_corpus_render_nebulae(11, first, sr, seconds, T.TS_F32, bad, pr, ar)
    T.ts_sync()
