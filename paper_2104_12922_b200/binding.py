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
_lib = None


class TsynthError(RuntimeError):
    pass


class _Out(C.Structure):
    _fields_ = [("audio", C.c_void_p), ("params_human", C.c_void_p)]


EXPORTS = ["ts_sample_params", "ts_render", "ts_render_host", "ts_corpus_render", "ts_corpus_is_test", "ts_num_samples", "ts_num_ticks", "ts_set_stream",
           "ts_default_nebula", "ts_set_nebula", "ts_workspace_bytes", "ts_last_error", "ts_sync", "ts_shutdown",
           "ts_set_timing", "ts_time_kernels", "ts_last_kernel_ms", "ts_last_stats", "ts_debug_noise_u32", "ts_debug_controls", "ts_render_controls",
           "ts_debug_phase"]


def lib_path() -> str:
    return _LIB_PATH


def lib():
    """Load libtsynth.so (built in-tree by paper_2104_12922_b200/build.py)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise TsynthError(f"{_LIB_PATH} is missing: run `python -m paper_2104_12922_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(_LIB_PATH)
    vp, u64, i32, f64 = C.c_void_p, C.c_uint64, C.c_int, C.c_double
    L.ts_sample_params.argtypes = [u64, u64, i32, vp]
    L.ts_render.argtypes = [vp, i32, i32, f64, _Out]
    L.ts_render_host.argtypes = [u64, u64, i32, i32, f64, vp, vp]
    L.ts_corpus_render.argtypes = [u64, u64, i32, i32, i32, f64, vp, vp, i32]
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
    L.ts_time_kernels.argtypes = [vp, i32, i32, f64, vp, i32, i32, vp]
    L.ts_last_stats.argtypes = [vp]
    L.ts_debug_noise_u32.argtypes = [vp, u64, i32, vp]
    L.ts_debug_controls.argtypes = [vp, i32, i32, f64, vp]
    L.ts_render_controls.argtypes = [vp, i32, i32, f64, vp]
    L.ts_debug_phase.argtypes = [vp, i32, i32, f64, i32, vp]
    _lib = L
    return L


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
    p = _dev_params(params)
    ms = (C.c_float * 2)()
    _use_current_stream(p.device)
    _check(lib().ts_time_kernels(C.c_void_p(p.data_ptr()), p.shape[0], sr, float(seconds), C.c_void_p(audio_ring.data_ptr()),
                                 int(audio_ring.shape[0]), reps, ms))
    return float(ms[0]), float(ms[1])


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
