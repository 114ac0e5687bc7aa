"""Builds the library in-tree with nvcc for sm_100a (cross-compiles without a GPU), twice from the same sources:
libtsynth.so          -- the product: what include/tsynth.h declares, nothing else;
libtsynth_measure.so  -- the product's sources + csrc/ts_measure.cu with -DTS_MEASURE: everything above plus the measurement
                         aids of include/tsynth_measure.h that bench.py's roofline numbers are made from."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtsynth.so")
LIB_MEASURE = os.path.join(HERE, "libtsynth_measure.so")
SOURCES = ["ts_api.cu", "ts_sample.cu", "ts_control.cu", "ts_audio.cu", "ts_mmd.cu"]
MEASURE_SOURCES = SOURCES + ["ts_measure.cu"]
HEADERS = [os.path.join(CSRC, "ts_common.cuh"), os.path.join(CSRC, "ts_math.cuh"), os.path.join(HERE, "..", "include", "tsynth.h"),
           os.path.join(HERE, "..", "include", "tsynth_measure.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]
TARGETS = ((LIB, SOURCES, []), (LIB_MEASURE, MEASURE_SOURCES, ["-DTS_MEASURE"]))


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def _stale(lib: str, sources) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in sources] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def stale() -> bool:
    return any(_stale(lib, src) for lib, src, _ in TARGETS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Both libraries, the two nvcc runs side by side.  -> path of libtsynth.so"""
    jobs = []
    for lib, sources, defs in TARGETS:
        if force or _stale(lib, sources):
            tmp = lib + f".tmp{os.getpid()}"
            cmd = [_nvcc()] + NVCC_FLAGS + defs + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + \
                  [os.path.join(CSRC, s) for s in sources]
            jobs.append((subprocess.Popen(cmd), cmd, tmp, lib))
    failed = None
    for proc, cmd, tmp, lib in jobs:
        if proc.wait() != 0:
            failed = failed or subprocess.CalledProcessError(proc.returncode, cmd)
        else:
            os.replace(tmp, lib)
    if failed:
        raise failed
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
