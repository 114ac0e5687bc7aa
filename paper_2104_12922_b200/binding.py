"""ctypes binding of libtsynth.so (include/tsynth.h).  Same names as the C entry points.

Marshalling only: PyTorch supplies device memory and the CUDA stream; every step of the path runs in
the library's kernels.  If the library is missing this module raises -- there is no fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

NPARAM = 78
R = 100
REC_FLOATS = 80  # sizeof(ts_voice) / 4: 78 params + 2 words of noise key
NEBULA_DTYPE = np.dtype([("lo", "<f8"), ("hi", "<f8"), ("curve", "<f8"), ("symmetric", "<i8")])

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtsynth.so")
_MEASURE_LIB_PATH = os.path.join(_HERE, "libtsynth_measure.so")
_lib = None
_measure = False


class TsynthError(RuntimeError):
    pass


class _Out(C.Structure):
    _fields_ = [("audio", C.c_void_p), ("params_human", C.c_void_p)]


EXPORTS = ["ts_sample_params", "ts_render", "ts_render_fmt", "ts_render_host", "ts_render_host_fmt", "ts_corpus_render",
           "ts_corpus_render_fmt", "ts_corpus_render_nebulae", "ts_corpus_open", "ts_corpus_next", "ts_corpus_close", "ts_corpus_is_test", "ts_num_samples",
           "ts_num_ticks", "ts_num_ticks_r", "ts_streaming_lanes", "ts_set_stream", "ts_default_nebula", "ts_set_nebula", "ts_workspace_bytes",
           "ts_last_error", "ts_sync", "ts_shutdown", "ts_set_timing", "ts_last_kernel_ms",
           "ts_last_stats", "ts_render_r", "ts_render_controls", "ts_render_controls_r", "ts_mmd_l1", "ts_mmd_l1_pairwise", "ts_mmd_l1_sorted", "ts_mmd_l1_static", "ts_debug_noise_u32", "ts_debug_controls",
           "ts_debug_phase"]
# include/tsynth_measure.h: only in libtsynth_measure.so (use_measure_build())
MEASURE_EXPORTS = ["ts_time_kernels", "ts_time_audio_lanes", "ts_time_fill", "ts_time_alu_bound", "ts_time_pipes"]
TS_F32, TS_F16, TS_BF16 = 0, 1, 2


class _CorpusCfg(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("B", C.c_int), ("sr", C.c_int), ("seconds", C.c_double), ("fmt", C.c_int),
                ("n_ring", C.c_int), ("d_audio_ring", C.c_void_p), ("d_params_ring", C.c_void_p)]


class _CorpusBatch(C.Structure):
    _fields_ = [("d_audio", C.c_void_p), ("d_params", C.c_void_p), ("batch_index", C.c_uint64), ("first_voice", C.c_uint64),
                ("is_test_first", C.c_int), ("is_test_last", C.c_int), ("slot", C.c_int)]


def lib_path() -> str:
    return _MEASURE_LIB_PATH if _measure else _LIB_PATH


def use_measure_build() -> None:
    """Make this process load libtsynth_measure.so INSTEAD of libtsynth.so: the same sources plus the measurement aids of
    include/tsynth_measure.h (the ts_time_* calls below), so that what bench.py times is the product's own code and the
    library state (nebula, workspaces, lanes) is one.  Must come before the first library call of the process."""
    global _measure
    if _lib is not None and not _measure:
        raise TsynthError("use_measure_build() must be called before the first library call (libtsynth.so is already loaded)")
    _measure = True


def lib():
    """Load libtsynth.so (built in-tree by paper_2104_12922_b200/build.py)."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise TsynthError(f"{path} is missing: run `python -m paper_2104_12922_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(path)
    vp, u64, i32, f64 = C.c_void_p, C.c_uint64, C.c_int, C.c_double
    L.ts_sample_params.argtypes = [u64, u64, i32, vp]
    L.ts_render.argtypes = [vp, i32, i32, f64, _Out]
    L.ts_render_fmt.argtypes = [vp, i32, i32, f64, i32, vp, vp]
    L.ts_render_host.argtypes = [u64, u64, i32, i32, f64, vp, vp]
    L.ts_render_host_fmt.argtypes = [u64, u64, i32, i32, f64, i32, vp, vp]
    L.ts_corpus_render.argtypes = [u64, u64, i32, i32, i32, f64, vp, vp, i32]
    L.ts_corpus_render_fmt.argtypes = [u64, u64, i32, i32, i32, f64, i32, vp, vp, i32]
    L.ts_corpus_render_nebulae.argtypes = [u64, u64, i32, i32, i32, f64, i32, vp, vp, vp, i32]
    L.ts_corpus_open.argtypes = [C.POINTER(_CorpusCfg), u64]
    L.ts_corpus_next.argtypes = [C.POINTER(_CorpusBatch)]
    L.ts_num_ticks_r.argtypes = [C.c_int64, i32]
    L.ts_num_ticks_r.restype = C.c_int64
    if _measure:
        L.ts_time_fill.argtypes = [vp, C.c_size_t, i32, vp]
        L.ts_time_audio_lanes.argtypes = [vp, i32, i32, f64, vp, i32, i32, vp]
        L.ts_time_alu_bound.argtypes = [i32, i32, vp]
        L.ts_time_pipes.argtypes = [vp]
        L.ts_time_kernels.argtypes = [vp, i32, i32, f64, vp, i32, i32, vp]
    L.ts_render_controls_r.argtypes = [vp, i32, i32, f64, i32, vp]
    L.ts_render_r.argtypes = [vp, i32, i32, f64, i32, vp]
    L.ts_mmd_l1.argtypes = [vp, vp, i32, i32, vp]
    L.ts_mmd_l1_pairwise.argtypes = [vp, vp, i32, i32, vp]
    L.ts_mmd_l1_sorted.argtypes = [vp, vp, i32, i32, vp]
    L.ts_mmd_l1_static.argtypes = [vp, vp, i32, i32, vp]
    L.ts_corpus_is_test.argtypes = [u64]
    L.ts_num_samples.argtypes = [i32, f64]
    L.ts_num_samples.restype = C.c_int64
    L.ts_num_ticks.argtypes = [C.c_int64]
    L.ts_num_ticks.restype = C.c_int64
    L.ts_set_stream.argtypes = [vp]
    L.ts_default_nebula.argtypes = [vp]
    L.ts_set_nebula.argtypes = [vp]
    L.ts_workspace_bytes.argtypes = [i32, i32, f64]
    L.ts_workspace_bytes.restype = C.c_size_t
    L.ts_last_error.restype = C.c_char_p
    L.ts_shutdown.restype = None
    L.ts_set_timing.argtypes = [i32]
    L.ts_last_kernel_ms.argtypes = [vp]
    L.ts_last_stats.argtypes = [vp]
    L.ts_debug_noise_u32.argtypes = [vp, u64, i32, vp]
    L.ts_debug_controls.argtypes = [vp, i32, i32, f64, vp]
    L.ts_render_controls.argtypes = [vp, i32, i32, f64, vp]
    L.ts_debug_phase.argtypes = [vp, i32, i32, f64, i32, vp]
    _lib = L
    return L


def _mlib():
    """The library, for a ts_time_* call: only the measure build has them."""
    if not _measure:
        raise TsynthError("the ts_time_* measurement aids are not in libtsynth.so: call use_measure_build() before the first "
                          "library call of the process (include/tsynth_measure.h)")
    return lib()


def _check(rc: int):
    if rc != 0:
        raise TsynthError(f"libtsynth error {rc}: {lib().ts_last_error().decode()}")


def _torch():
    import torch
    return torch


def _use_current_stream(device):
    torch = _torch()
    _check(lib().ts_set_stream(C.c_void_p(torch.cuda.current_stream(device).cuda_stream)))


def _dev_params(params):
    torch = _torch()
    if not (params.is_cuda and params.dtype == torch.float32 and params.dim() == 2
            and params.shape[1] == REC_FLOATS and params.is_contiguous()):
        raise TsynthError("params must be a contiguous CUDA float32 tensor [B, 80] (ts_voice records)")
    return params


# ------------------------------------------------------------------------------------------ host helpers
def ts_corpus_is_test(g: int) -> bool:
    return bool(lib().ts_corpus_is_test(g))


def ts_num_samples(sr: int, seconds: float) -> int:
    return lib().ts_num_samples(sr, seconds)


def ts_num_ticks(N: int) -> int:
    return lib().ts_num_ticks(N)


def ts_default_nebula() -> np.ndarray:
    neb = np.zeros(NPARAM, dtype=NEBULA_DTYPE)
    _check(lib().ts_default_nebula(neb.ctypes.data_as(C.c_void_p)))
    return neb


def ts_set_nebula(neb) -> None:
    if neb is None:
        _check(lib().ts_set_nebula(None))
        return
    neb = np.ascontiguousarray(neb, dtype=NEBULA_DTYPE)
    if neb.shape != (NPARAM,):
        raise TsynthError("nebula must have 78 entries")
    _check(lib().ts_set_nebula(neb.ctypes.data_as(C.c_void_p)))


def ts_streaming_lanes() -> int:
    return lib().ts_streaming_lanes()


def ts_workspace_bytes(B: int, sr: int, seconds: float) -> int:
    return lib().ts_workspace_bytes(B, sr, seconds)


def ts_set_stream(cuda_stream: int | None) -> None:
    _check(lib().ts_set_stream(C.c_void_p(cuda_stream or 0)))


def ts_sync() -> None:
    _check(lib().ts_sync())


def ts_shutdown() -> None:
    lib().ts_shutdown()


def ts_set_timing(enable: bool) -> None:
    _check(lib().ts_set_timing(int(enable)))


def ts_last_kernel_ms():
    ms = (C.c_float * 2)()
    _check(lib().ts_last_kernel_ms(ms))
    return float(ms[0]), float(ms[1])


def ts_time_kernels(params, sr: int, seconds: float, audio_ring, reps: int):
    """-> (control ms, audio ms) per launch, averaged over `reps` back-to-back launches of each kernel."""
    _mlib()  # refuse before touching CUDA if this process runs the product build
    p = _dev_params(params)
    ms = (C.c_float * 2)()
    _use_current_stream(p.device)
    _check(_mlib().ts_time_kernels(C.c_void_p(p.data_ptr()), p.shape[0], sr, float(seconds), C.c_void_p(audio_ring.data_ptr()),
                                 int(audio_ring.shape[0]), reps, ms))
    return float(ms[0]), float(ms[1])


def ts_time_audio_lanes(params, sr: int, seconds: float, audio_ring, reps: int) -> float:
    """-> ms per audio launch when launches rotate over the lanes' audio streams (inverse throughput, not a duration)."""
    _mlib()  # refuse before touching CUDA if this process runs the product build
    p = _dev_params(params)
    ms = C.c_float()
    _use_current_stream(p.device)
    _check(_mlib().ts_time_audio_lanes(C.c_void_p(p.data_ptr()), p.shape[0], sr, float(seconds), C.c_void_p(audio_ring.data_ptr()),
                                           int(audio_ring.shape[0]), reps, C.byref(ms)))
    return float(ms.value)


def ts_last_stats():
    st = (C.c_int64 * 3)()
    _check(lib().ts_last_stats(st))
    return {"launches": int(st[0]), "chunks": int(st[1]), "active_samples": int(st[2])}


# ------------------------------------------------------------------------------------------ device calls
def ts_sample_params(seed: int, batch_index: int, B: int, device="cuda:0", out=None):
    """-> CUDA float32 tensor [B, 80]: ts_voice records (u[78] then the two noise-key words, bit-cast)."""
    torch = _torch()
    if out is None:
        out = torch.empty((B, REC_FLOATS), dtype=torch.float32, device=device)
    _dev_params(out)
    _use_current_stream(out.device)
    _check(lib().ts_sample_params(seed, batch_index, B, C.c_void_p(out.data_ptr())))
    return out


def ts_render(params, sr: int, seconds: float, out=None, want_human: bool = False):
    """params: [B, 80] records on the GPU -> audio [B, N] fp32 (and params_human [B, 78] if asked)."""
    torch = _torch()
    p = _dev_params(params)
    B = p.shape[0]
    if ts_workspace_bytes(B, sr, float(seconds)) == 0:      # the library's own size check (TS_EINVAL)
        raise TsynthError(f"libtsynth error -1: {lib().ts_last_error().decode()}")
    N = ts_num_samples(sr, seconds)
    if out is None:
        out = torch.empty((B, N), dtype=torch.float32, device=p.device)
    elif not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and tuple(out.shape) == (B, N)):
        raise TsynthError("out must be a contiguous CUDA float32 tensor [B, N]")
    human = torch.empty((B, NPARAM), dtype=torch.float32, device=p.device) if want_human else None
    _use_current_stream(p.device)
    o = _Out(C.c_void_p(out.data_ptr()), C.c_void_p(human.data_ptr()) if want_human else None)
    _check(lib().ts_render(C.c_void_p(p.data_ptr()), B, sr, float(seconds), o))
    return (out, human) if want_human else out


def ts_render_host(seed: int, batch_index: int, B: int, sr: int, seconds: float, host_audio=None, host_params=None):
    """End to end with HOST buffers (pinned torch CPU tensors or numpy arrays): sample + render + D2H."""
    torch = _torch()
    N = ts_num_samples(sr, seconds)
    if host_audio is None:
        host_audio = torch.empty((B, N), dtype=torch.float32, pin_memory=True)
    ap = host_audio.data_ptr() if hasattr(host_audio, "data_ptr") else host_audio.ctypes.data
    pp = None
    if host_params is not None:
        pp = host_params.data_ptr() if hasattr(host_params, "data_ptr") else host_params.ctypes.data
    _use_current_stream(torch.device("cuda", torch.cuda.current_device()))
    _check(lib().ts_render_host(seed, batch_index, B, sr, float(seconds), C.c_void_p(ap), C.c_void_p(pp) if pp else None))
    return host_audio


def ts_corpus_render(seed: int, first_batch: int, n_batches: int, sr: int, seconds: float, params_ring, audio_ring):
    """Streams n_batches consecutive batches into the rings: params_ring [R, B, 80], audio_ring [R, B, N] (CUDA fp32)."""
    torch = _torch()
    if not (params_ring.is_cuda and params_ring.dtype == torch.float32 and params_ring.dim() == 3
            and params_ring.shape[2] == REC_FLOATS and params_ring.is_contiguous()):
        raise TsynthError("params_ring must be a contiguous CUDA float32 tensor [R, B, 80]")
    R_, B = int(params_ring.shape[0]), int(params_ring.shape[1])
    N = ts_num_samples(sr, seconds)
    if not (audio_ring.is_cuda and audio_ring.dtype == torch.float32 and audio_ring.is_contiguous()
            and tuple(audio_ring.shape) == (R_, B, N)):
        raise TsynthError("audio_ring must be a contiguous CUDA float32 tensor [R, B, N]")
    _use_current_stream(params_ring.device)
    _check(lib().ts_corpus_render(seed, first_batch, n_batches, B, sr, float(seconds), C.c_void_p(params_ring.data_ptr()),
                                  C.c_void_p(audio_ring.data_ptr()), R_))
    return audio_ring


def _fmt_dtype(fmt: int):
    torch = _torch()
    return {TS_F32: torch.float32, TS_F16: torch.float16, TS_BF16: torch.bfloat16}[fmt]


def ts_num_ticks_r(N: int, R: int) -> int:
    return lib().ts_num_ticks_r(N, R)


def ts_render_fmt(params, sr: int, seconds: float, fmt: int, out=None):
    """ts_render with the output format chosen per call -> audio [B, N] in float32 / float16 / bfloat16."""
    torch = _torch()
    p = _dev_params(params)
    B = p.shape[0]
    N = ts_num_samples(sr, seconds)
    dt = _fmt_dtype(fmt)
    if out is None:
        out = torch.empty((B, N), dtype=dt, device=p.device)
    elif not (out.is_cuda and out.dtype == dt and out.is_contiguous() and tuple(out.shape) == (B, N)):
        raise TsynthError("out must be a contiguous CUDA tensor [B, N] of the chosen format")
    _use_current_stream(p.device)
    _check(lib().ts_render_fmt(C.c_void_p(p.data_ptr()), B, sr, float(seconds), fmt, C.c_void_p(out.data_ptr()), None))
    return out


def ts_render_host_fmt(seed: int, batch_index: int, B: int, sr: int, seconds: float, fmt: int, host_audio=None, host_params=None):
    """End to end with HOST buffers in the chosen format (pinned torch CPU tensors): sample + render + D2H."""
    torch = _torch()
    N = ts_num_samples(sr, seconds)
    if host_audio is None:
        host_audio = torch.empty((B, N), dtype=_fmt_dtype(fmt), pin_memory=True)
    pp = host_params.data_ptr() if host_params is not None else None
    _use_current_stream(torch.device("cuda", torch.cuda.current_device()))
    _check(lib().ts_render_host_fmt(seed, batch_index, B, sr, float(seconds), fmt, C.c_void_p(host_audio.data_ptr()),
                                    C.c_void_p(pp) if pp else None))
    return host_audio


def ts_corpus_render_fmt(seed: int, first_batch: int, n_batches: int, sr: int, seconds: float, fmt: int, params_ring, audio_ring):
    """ts_corpus_render with the output format chosen per call; audio_ring [R, B, N] in that format."""
    R_, B = int(params_ring.shape[0]), int(params_ring.shape[1])
    N = ts_num_samples(sr, seconds)
    if not (audio_ring.is_cuda and audio_ring.dtype == _fmt_dtype(fmt) and audio_ring.is_contiguous()
            and tuple(audio_ring.shape) == (R_, B, N)):
        raise TsynthError("audio_ring must be a contiguous CUDA tensor [R, B, N] of the chosen format")
    _use_current_stream(params_ring.device)
    _check(lib().ts_corpus_render_fmt(seed, first_batch, n_batches, B, sr, float(seconds), fmt, C.c_void_p(params_ring.data_ptr()),
                                      C.c_void_p(audio_ring.data_ptr()), R_))
    return audio_ring


def ts_corpus_render_nebulae(seed: int, first_batch: int, sr: int, seconds: float, fmt: int, nebulae, params_ring, audio_ring):
    """One nebula per batch: nebulae is a sequence / array [n_batches, 78] of NEBULA_DTYPE; batch i of the stream is mapped
    with table i.  audio_ring [R, B, N] in fmt, params_ring [R, B, 80] fp32."""
    tabs = np.ascontiguousarray(nebulae, dtype=NEBULA_DTYPE)
    if tabs.ndim != 2 or tabs.shape[1] != NPARAM or tabs.shape[0] < 1:
        raise TsynthError("nebulae must be [n_batches, 78]")
    R_, B = int(params_ring.shape[0]), int(params_ring.shape[1])
    N = ts_num_samples(sr, seconds)
    if not (params_ring.is_cuda and params_ring.is_contiguous() and params_ring.shape[2] == REC_FLOATS):
        raise TsynthError("params_ring must be a contiguous CUDA float32 tensor [R, B, 80]")
    if not (audio_ring.is_cuda and audio_ring.dtype == _fmt_dtype(fmt) and audio_ring.is_contiguous()
            and tuple(audio_ring.shape) == (R_, B, N)):
        raise TsynthError("audio_ring must be a contiguous CUDA tensor [R, B, N] of the chosen format")
    _use_current_stream(params_ring.device)
    _check(lib().ts_corpus_render_nebulae(seed, first_batch, int(tabs.shape[0]), B, sr, float(seconds), fmt,
                                          tabs.ctypes.data_as(C.c_void_p), C.c_void_p(params_ring.data_ptr()),
                                          C.c_void_p(audio_ring.data_ptr()), R_))
    return audio_ring


_corpus_rings = None


def ts_corpus_open(seed: int, first_batch: int, sr: int, seconds: float, fmt: int, params_ring, audio_ring) -> None:
    """Opens the streaming iterator over the caller's rings: params_ring [R, B, 80] fp32, audio_ring [R, B, N] in fmt."""
    global _corpus_rings
    R_, B = int(params_ring.shape[0]), int(params_ring.shape[1])
    N = ts_num_samples(sr, seconds)
    if not (params_ring.is_cuda and params_ring.is_contiguous() and params_ring.shape[2] == REC_FLOATS):
        raise TsynthError("params_ring must be a contiguous CUDA float32 tensor [R, B, 80]")
    if not (audio_ring.is_cuda and audio_ring.dtype == _fmt_dtype(fmt) and audio_ring.is_contiguous()
            and tuple(audio_ring.shape) == (R_, B, N)):
        raise TsynthError("audio_ring must be a contiguous CUDA tensor [R, B, N] of the chosen format")
    cfg = _CorpusCfg(seed, B, sr, float(seconds), fmt, R_, audio_ring.data_ptr(), params_ring.data_ptr())
    _use_current_stream(params_ring.device)
    _check(lib().ts_corpus_open(C.byref(cfg), first_batch))
    _corpus_rings = (params_ring, audio_ring)


def ts_corpus_next():
    """-> dict(audio [B, N] view of the ring slot, params [B, 80] view, batch_index, first_voice, is_test_first,
    is_test_last, slot).  The current torch stream waits for the batch; consume it there before the next call."""
    if _corpus_rings is None:
        raise TsynthError("no corpus iterator is open")
    params_ring, audio_ring = _corpus_rings
    b = _CorpusBatch()
    _use_current_stream(params_ring.device)
    _check(lib().ts_corpus_next(C.byref(b)))
    assert b.d_audio == audio_ring[b.slot].data_ptr() and b.d_params == params_ring[b.slot].data_ptr()
    return {"audio": audio_ring[b.slot], "params": params_ring[b.slot], "batch_index": int(b.batch_index),
            "first_voice": int(b.first_voice), "is_test_first": bool(b.is_test_first), "is_test_last": bool(b.is_test_last),
            "slot": int(b.slot)}


def ts_corpus_close() -> None:
    global _corpus_rings
    _check(lib().ts_corpus_close())
    _corpus_rings = None


def ts_time_fill(buf, reps: int) -> float:
    """-> ms per launch of a store-only fill of `buf` (a CUDA tensor)."""
    _mlib()  # refuse before touching CUDA if this process runs the product build
    ms = C.c_float()
    _use_current_stream(buf.device)
    _check(_mlib().ts_time_fill(C.c_void_p(buf.data_ptr()), buf.numel() * buf.element_size(), reps, C.byref(ms)))
    return float(ms.value)


def ts_time_alu_bound(fastsin: bool, reps: int = 64) -> float:
    """-> audible samples/s the SM pipes sustain on the audio kernel's own sample loop (no memory, no CTA turnover)."""
    _mlib()  # refuse before touching CUDA if this process runs the product build
    v = C.c_double()
    _use_current_stream(_torch().device("cuda", _torch().cuda.current_device()))
    _check(_mlib().ts_time_alu_bound(int(fastsin), reps, C.byref(v)))
    return float(v.value)


PIPE_NAMES = ["FFMA", "FFMA2", "IMAD.WIDE.U32", "LOP3", "DFMA", "MUFU.SIN+FMUL", "MUFU.EX2", "I2FP"]


def ts_time_pipes() -> dict:
    """-> {instruction kind: cycles per warp instruction per SM sub-partition}, each kind issued alone."""
    _mlib()  # refuse before touching CUDA if this process runs the product build
    r = (C.c_double * 8)()
    _use_current_stream(_torch().device("cuda", _torch().cuda.current_device()))
    _check(_mlib().ts_time_pipes(r))
    return {n: float(r[i]) for i, n in enumerate(PIPE_NAMES)}


def ts_render_r(params, sr: int, seconds: float, R: int):
    """ts_render with the tick spacing chosen per call (R = 100, or R = 1: audio-rate control) -> fp32 audio [B, N]."""
    torch = _torch()
    p = _dev_params(params)
    B = p.shape[0]
    N = ts_num_samples(sr, seconds)
    out = torch.empty((B, N), dtype=torch.float32, device=p.device)
    _use_current_stream(p.device)
    _check(lib().ts_render_r(C.c_void_p(p.data_ptr()), B, sr, float(seconds), R, C.c_void_p(out.data_ptr())))
    return out


def ts_render_controls_r(params, sr: int, seconds: float, R: int):
    """-> CUDA float64 tensor [B, 5, K_R]: the modulation-mixer rows with one control tick every R samples."""
    torch = _torch()
    p = _dev_params(params)
    B = p.shape[0]
    K = ts_num_ticks_r(ts_num_samples(sr, seconds), R)
    out = torch.empty((B, 5, K), dtype=torch.float64, device=p.device)
    _use_current_stream(p.device)
    _check(lib().ts_render_controls_r(C.c_void_p(p.data_ptr()), B, sr, float(seconds), R, C.c_void_p(out.data_ptr())))
    return out


def ts_mmd_l1(x, y, form: str = "auto"):
    """x, y: CUDA float32 [n, d] -> CUDA float64 [4]: MMD (Eq. 2), sum |x_i - y_j|_1, sum |x_i - x_j|_1, sum |y_i - y_j|_1.
    form: "auto" (ts_mmd_l1: the faster form at this n), "pairwise" (ts_mmd_l1_pairwise) or "sorted" (ts_mmd_l1_sorted)."""
    torch = _torch()
    if not (x.is_cuda and y.is_cuda and x.dtype == torch.float32 and y.dtype == torch.float32 and x.is_contiguous()
            and y.is_contiguous() and x.dim() == 2 and tuple(x.shape) == tuple(y.shape)):
        raise TsynthError("x and y must be contiguous CUDA float32 tensors of the same shape [n, d]")
    out = torch.empty(4, dtype=torch.float64, device=x.device)
    _use_current_stream(x.device)
    fn = {"auto": lib().ts_mmd_l1, "pairwise": lib().ts_mmd_l1_pairwise, "sorted": lib().ts_mmd_l1_sorted}[form]
    _check(fn(C.c_void_p(x.data_ptr()), C.c_void_p(y.data_ptr()), int(x.shape[0]), int(x.shape[1]), C.c_void_p(out.data_ptr())))
    return out


MMD_STATIC_MAX_PARTIALS = 32768  # TS_MMD_STATIC_MAX_PARTIALS


def ts_mmd_l1_static(x, y, out=None):
    """ts_mmd_l1 without any device allocation inside the library: for hosts that cannot call cudaMalloc when the call is
    made (all of the GPU's memory already belongs to another allocator, a real-time loop that cannot afford cudaMalloc's
    device-wide synchronisation, a host that forbids allocation after start-up).  Same kernels and same bits as
    ts_mmd_l1(x, y); the scratch is a 256 KB array inside the library's device image, so n <= 4032 and d <= 10922
    (TsynthError beyond that).  Pass a preallocated CUDA float64 [4] tensor as `out` to keep this wrapper from asking torch
    for one.  All calls share the scratch: keep them on one stream.  Make the first call (it looks up the array's device
    address) during start-up."""
    torch = _torch()
    if not (x.is_cuda and y.is_cuda and x.dtype == torch.float32 and y.dtype == torch.float32 and x.is_contiguous()
            and y.is_contiguous() and x.dim() == 2 and tuple(x.shape) == tuple(y.shape)):
        raise TsynthError("x and y must be contiguous CUDA float32 tensors of the same shape [n, d]")
    if out is None:
        out = torch.empty(4, dtype=torch.float64, device=x.device)
    elif not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 4 and out.device == x.device):
        raise TsynthError("out must be a contiguous CUDA float64 tensor of 4 elements on the device of x")
    _use_current_stream(x.device)
    _check(lib().ts_mmd_l1_static(C.c_void_p(x.data_ptr()), C.c_void_p(y.data_ptr()), int(x.shape[0]), int(x.shape[1]),
                                  C.c_void_p(out.data_ptr())))
    return out


def ts_debug_noise_u32(key, n0: int, count: int, device="cuda:0"):
    torch = _torch()
    k = (C.c_uint32 * 2)(int(key[0]), int(key[1]))
    out = torch.empty(count, dtype=torch.int32, device=device)
    _use_current_stream(out.device)
    _check(lib().ts_debug_noise_u32(k, n0, count, C.c_void_p(out.data_ptr())))
    return out


def ts_debug_controls(params, sr: int, seconds: float):
    torch = _torch()
    p = _dev_params(params)
    B = p.shape[0]
    K = ts_num_ticks(ts_num_samples(sr, seconds))
    out = torch.empty((B, 5, K), dtype=torch.float64, device=p.device)
    _use_current_stream(p.device)
    _check(lib().ts_debug_controls(C.c_void_p(p.data_ptr()), B, sr, float(seconds), C.c_void_p(out.data_ptr())))
    return out


def ts_render_controls(params, sr: int, seconds: float):
    """-> CUDA float64 tensor [B, 5, K]: the modulation-mixer rows at the control ticks (S5..S7)."""
    torch = _torch()
    p = _dev_params(params)
    B = p.shape[0]
    K = ts_num_ticks(ts_num_samples(sr, seconds))
    out = torch.empty((B, 5, K), dtype=torch.float64, device=p.device)
    _use_current_stream(p.device)
    _check(lib().ts_render_controls(C.c_void_p(p.data_ptr()), B, sr, float(seconds), C.c_void_p(out.data_ptr())))
    return out


def ts_debug_phase(params, sr: int, seconds: float, vco: int):
    torch = _torch()
    p = _dev_params(params)
    B = p.shape[0]
    N = ts_num_samples(sr, seconds)
    out = torch.empty((B, N), dtype=torch.float64, device=p.device)
    _use_current_stream(p.device)
    _check(lib().ts_debug_phase(C.c_void_p(p.data_ptr()), B, sr, float(seconds), vco, C.c_void_p(out.data_ptr())))
    return out
