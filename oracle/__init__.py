"""ORACLE (test infrastructure, not the product): ctypes loader for oracle/ts_oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2104_12922_b200 and shares no code with
the CUDA path.  See the header of ts_oracle.c for what each function follows and how it is pinned.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ts_oracle.c")
_LIB = os.path.join(_HERE, "libts_oracle.so")

NPARAM = 78
R = 100


class Range(C.Structure):
    _fields_ = [("lo", C.c_double), ("hi", C.c_double), ("curve", C.c_double), ("symmetric", C.c_int64)]


Nebula = Range * NPARAM


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off (one rounding per written operation, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u32p, f32p, f64p = C.POINTER(C.c_uint32), C.POINTER(C.c_float), C.POINTER(C.c_double)
        L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.orc_sample_params.argtypes = [C.c_uint64, C.c_uint64, f32p, u32p]
        L.orc_default_nebula.argtypes = [C.POINTER(Range)]
        L.orc_map.argtypes = [C.c_double] * 4 + [C.c_int64]
        L.orc_map.restype = C.c_double
        L.orc_map_all.argtypes = [f32p, C.POINTER(Range), f64p]
        L.orc_adsr.argtypes = [C.c_double] * 7
        L.orc_adsr.restype = C.c_double
        L.orc_num_ticks.argtypes = [C.c_int64]
        L.orc_num_ticks.restype = C.c_int64
        L.orc_lfo_shapes.argtypes = [C.c_double, f64p]
        L.orc_controls.argtypes = [f64p, C.c_int, C.c_int64, f64p, f64p, f64p]
        L.orc_upsample.argtypes = [f64p, C.c_int64]
        L.orc_upsample.restype = C.c_double
        L.orc_squaresaw.argtypes = [C.c_double] * 3
        L.orc_squaresaw.restype = C.c_double
        L.orc_squaresaw_k.argtypes = [C.c_double] * 2
        L.orc_squaresaw_k.restype = C.c_double
        L.orc_noise_word.argtypes = [u32p, C.c_uint64]
        L.orc_noise_word.restype = C.c_uint32
        L.orc_noise_value.argtypes = [C.c_uint32]
        L.orc_noise_value.restype = C.c_double
        L.orc_render_voice.argtypes = [f32p, u32p, C.POINTER(Range), C.c_int, C.c_int64, f64p, f64p, f64p, f64p]
        L.orc_render_voice.restype = C.c_int
        L.orc_num_samples.argtypes = [C.c_int, C.c_double]
        L.orc_num_samples.restype = C.c_int64
        L.orc_num_ticks_r.argtypes = [C.c_int64, C.c_int]
        L.orc_num_ticks_r.restype = C.c_int64
        L.orc_controls_r.argtypes = [f64p, C.c_int, C.c_int64, C.c_int, f64p, f64p, f64p]
        L.orc_upsample_r.argtypes = [f64p, C.c_int64, C.c_int]
        L.orc_upsample_r.restype = C.c_double
        L.orc_render_voice_r.argtypes = [f32p, u32p, C.POINTER(Range), C.c_int, C.c_int64, C.c_int, f64p, f64p, f64p, f64p]
        L.orc_render_voice_r.restype = C.c_int
        L.orc_mmd_l1.argtypes = [f64p, f64p, C.c_int, C.c_int, f64p]
        L.orc_mmd_l1.restype = C.c_double
        L.orc_corpus_is_test.argtypes = [C.c_uint64]
        _lib = L
    return _lib


def _p(a, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def sample_params(seed: int, batch_index: int, B: int):
    """-> (u float32 [B,78], noise_key uint32 [B,2]); global voice index g = batch_index*B + b (D3)."""
    u = np.empty((B, NPARAM), dtype=np.float32)
    nk = np.empty((B, 2), dtype=np.uint32)
    for b in range(B):
        lib().orc_sample_params(seed, batch_index * B + b, _p(u[b], C.c_float), _p(nk[b], C.c_uint32))
    return u, nk


def default_nebula() -> np.ndarray:
    """-> structured array [78] with fields lo, hi, curve (f8) and symmetric (i8)."""
    neb = np.zeros(NPARAM, dtype=NEBULA_DTYPE)
    lib().orc_default_nebula(neb.ctypes.data_as(C.POINTER(Range)))
    return neb


NEBULA_DTYPE = np.dtype([("lo", "<f8"), ("hi", "<f8"), ("curve", "<f8"), ("symmetric", "<i8")])


def _neb_ptr(neb):
    neb = np.ascontiguousarray(neb, dtype=NEBULA_DTYPE)
    assert neb.shape == (NPARAM,)
    return neb, neb.ctypes.data_as(C.POINTER(Range))


def map_param(u, lo, hi, curve, symmetric) -> float:
    return lib().orc_map(float(u), float(lo), float(hi), float(curve), int(symmetric))


def map_all(u, neb=None) -> np.ndarray:
    neb, nptr = _neb_ptr(default_nebula() if neb is None else neb)
    u = np.ascontiguousarray(u, dtype=np.float32)
    h = np.empty(NPARAM, dtype=np.float64)
    lib().orc_map_all(_p(u, C.c_float), nptr, _p(h, C.c_double))
    return h


def adsr(t, A, Dc, S, Rl, alpha, D) -> float:
    return lib().orc_adsr(float(t), float(A), float(Dc), float(S), float(Rl), float(alpha), float(D))


def corpus_is_test(g: int) -> bool:
    return bool(lib().orc_corpus_is_test(g))


def num_ticks_r(N: int, R: int) -> int:
    return lib().orc_num_ticks_r(N, R)


def controls_r(h, sr: int, N: int, R: int):
    """human params h[78], one control tick every R samples -> (E[6,K], L[2,K], M[5,K]), K = ceil(N/R) + 1."""
    h = np.ascontiguousarray(h, dtype=np.float64)
    K = num_ticks_r(N, R)
    E = np.empty((6, K)); Lf = np.empty((2, K)); M = np.empty((5, K))
    lib().orc_controls_r(_p(h, C.c_double), sr, N, R, _p(E, C.c_double), _p(Lf, C.c_double), _p(M, C.c_double))
    return E, Lf, M


def upsample_r(Cs, n: int, R: int) -> float:
    Cs = np.ascontiguousarray(Cs, dtype=np.float64)
    return lib().orc_upsample_r(_p(Cs, C.c_double), n, R)


def render_voice_r(u, noise_key, sr: int, N: int, R: int, neb=None, want_phase: bool = False):
    """One voice with one control tick every R samples -> dict(audio f64[N], phase1, phase2)."""
    neb, nptr = _neb_ptr(default_nebula() if neb is None else neb)
    u = np.ascontiguousarray(u, dtype=np.float32)
    k = np.ascontiguousarray(noise_key, dtype=np.uint32)
    audio = np.empty(N, dtype=np.float64)
    p1 = np.empty(N, dtype=np.float64) if want_phase else None
    p2 = np.empty(N, dtype=np.float64) if want_phase else None
    null = C.POINTER(C.c_double)()
    rc = lib().orc_render_voice_r(_p(u, C.c_float), _p(k, C.c_uint32), nptr, sr, N, R, _p(audio, C.c_double),
                                  _p(p1, C.c_double) if want_phase else null, _p(p2, C.c_double) if want_phase else null, null)
    if rc != 0:
        raise MemoryError("orc_render_voice_r")
    return {"audio": audio, "phase1": p1, "phase2": p2}


def mmd_l1(X, Y):
    """Eq. 2 with the l1 core distance -> (MMD, [sum d(x,y), sum d(x,x), sum d(y,y)]); X, Y: [n, d]."""
    X = np.ascontiguousarray(X, dtype=np.float64)
    Y = np.ascontiguousarray(Y, dtype=np.float64)
    assert X.shape == Y.shape and X.ndim == 2
    sums = np.empty(3, dtype=np.float64)
    v = lib().orc_mmd_l1(_p(X, C.c_double), _p(Y, C.c_double), X.shape[0], X.shape[1], _p(sums, C.c_double))
    return v, sums


def round_bf16(x) -> np.ndarray:
    """fp64/fp32 values -> the nearest bfloat16 (round to nearest even, through fp32 as the GPU path does), as float32."""
    b = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    b = (b + 0x7FFF + ((b >> 16) & 1)) & 0xFFFF0000
    return b.astype(np.uint32).view(np.float32)


def round_f16(x) -> np.ndarray:
    """fp64/fp32 values -> the nearest IEEE half (round to nearest even, through fp32 as the GPU path does), as float32."""
    return np.ascontiguousarray(x, dtype=np.float32).astype(np.float16).astype(np.float32)


def num_ticks(N: int) -> int:
    return lib().orc_num_ticks(N)


def num_samples(sr: int, seconds: float) -> int:
    return lib().orc_num_samples(sr, seconds)


def lfo_shapes(p: float) -> np.ndarray:
    sh = np.empty(5, dtype=np.float64)
    lib().orc_lfo_shapes(float(p), _p(sh, C.c_double))
    return sh


def controls(h, sr: int, N: int):
    """human params h[78] -> (E[6,K], L[2,K], M[5,K])."""
    h = np.ascontiguousarray(h, dtype=np.float64)
    K = num_ticks(N)
    E = np.empty((6, K)); Lf = np.empty((2, K)); M = np.empty((5, K))
    lib().orc_controls(_p(h, C.c_double), sr, N, _p(E, C.c_double), _p(Lf, C.c_double), _p(M, C.c_double))
    return E, Lf, M


def upsample(Cs, n: int) -> float:
    Cs = np.ascontiguousarray(Cs, dtype=np.float64)
    return lib().orc_upsample(_p(Cs, C.c_double), n)


def squaresaw(theta, k, s) -> float:
    return lib().orc_squaresaw(float(theta), float(k), float(s))


def squaresaw_k(midi, tune2) -> float:
    return lib().orc_squaresaw_k(float(midi), float(tune2))


def noise_word(noise_key, n: int) -> int:
    k = np.ascontiguousarray(noise_key, dtype=np.uint32)
    return lib().orc_noise_word(_p(k, C.c_uint32), n)


def noise_value(x: int) -> float:
    return lib().orc_noise_value(x)


def render_voice(u, noise_key, sr: int, N: int, neb=None, want_phase: bool = False, want_human: bool = False):
    """One voice -> dict(audio f64[N], phase1, phase2 (f64[N] or None), human (f64[78] or None))."""
    neb, nptr = _neb_ptr(default_nebula() if neb is None else neb)
    u = np.ascontiguousarray(u, dtype=np.float32)
    k = np.ascontiguousarray(noise_key, dtype=np.uint32)
    audio = np.empty(N, dtype=np.float64)
    p1 = np.empty(N, dtype=np.float64) if want_phase else None
    p2 = np.empty(N, dtype=np.float64) if want_phase else None
    hm = np.empty(NPARAM, dtype=np.float64) if want_human else None
    null = C.POINTER(C.c_double)()
    rc = lib().orc_render_voice(
        _p(u, C.c_float), _p(k, C.c_uint32), nptr, sr, N, _p(audio, C.c_double),
        _p(p1, C.c_double) if want_phase else null, _p(p2, C.c_double) if want_phase else null,
        _p(hm, C.c_double) if want_human else null)
    if rc != 0:
        raise MemoryError("orc_render_voice")
    return {"audio": audio, "phase1": p1, "phase2": p2, "human": hm}


def render_batch(u, noise_key, sr: int, N: int, neb=None, threads: int | None = None, dtype=np.float64, out=None):
    """Voices are independent: render rows on a thread pool (ctypes releases the GIL).
    -> audio [B,N] in `dtype` (float64 = the oracle's own values)."""
    u = np.ascontiguousarray(u, dtype=np.float32)
    B = u.shape[0]
    if out is None:
        out = np.empty((B, N), dtype=dtype)
    threads = threads or os.cpu_count() or 1

    def one(b):
        out[b] = render_voice(u[b], noise_key[b], sr, N, neb)["audio"]

    if threads == 1:
        for b in range(B):
            one(b)
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(one, range(B)))
    return out
