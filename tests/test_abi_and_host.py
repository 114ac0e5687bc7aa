"""CPU-only checks of the boundary and host logic: the C-ABI library builds, loads and exports every
symbol include/tsynth.h declares (no compute calls: there is no GPU here), host-side helpers agree with
the oracle, and the workload generators are deterministic."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle as O
from paper_2104_12922_b200 import binding, build, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build.build()
    return binding.lib()


def declared_symbols(header="tsynth.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ts_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(L):
    names = declared_symbols()
    assert len(names) >= 18
    for n in names:
        assert hasattr(L, n), n
    assert sorted(binding.EXPORTS) == names


def test_measurement_aids_live_in_their_own_header_and_library(L):
    """include/tsynth_measure.h <-> libtsynth_measure.so (the same sources + ts_measure.cu with -DTS_MEASURE): that build
    exports both headers' symbols; the product library exports none of the measurement aids and no bench kernel."""
    aids = declared_symbols("tsynth_measure.h")
    assert aids == sorted(binding.MEASURE_EXPORTS) and len(aids) == 5
    assert not set(aids) & set(declared_symbols())
    M = ctypes.CDLL(build.LIB_MEASURE)
    for n in aids + declared_symbols():
        assert hasattr(M, n), n
    for n in aids:
        assert not hasattr(L, n), n
    blob = open(build.LIB, "rb").read()
    for needle in (b"ts_time_", b"ts_body_bench_kernel", b"ts_pipe_kernel", b"ts_fill_kernel"):
        assert needle not in blob, needle
    with pytest.raises(binding.TsynthError, match="use_measure_build"):
        binding.ts_time_pipes()                               # this process runs the product build


def test_struct_sizes_match_header():
    assert ctypes.sizeof(ctypes.c_float) * 80 == 320
    assert binding.NEBULA_DTYPE.itemsize == 32
    assert binding.REC_FLOATS * 4 == 320


def test_host_helpers_match_oracle(L):
    for sr, s in [(44100, 1.0), (44100, 4.0), (48000, 30.0), (44100, 0.0123), (44101, 0.3), (8000, 1.0)]:
        N = binding.ts_num_samples(sr, s)
        assert N == O.num_samples(sr, s)
        assert binding.ts_num_ticks(N) == O.num_ticks(N)
    g, o = binding.ts_default_nebula(), O.default_nebula()
    for f in ("lo", "hi", "curve", "symmetric"):
        assert np.array_equal(g[f], o[f]), f          # same table on both sides, as doubles


def test_workspace_is_bounded_for_l2(L):
    # the control table is chunked over voices so that it stays L2-resident
    for name, wl in W.WORKLOADS.items():
        ws = binding.ts_workspace_bytes(wl.B, wl.sr, wl.seconds)
        assert 0 < ws <= (64 << 20), (name, ws)
    assert binding.ts_workspace_bytes(0, 44100, 1.0) == 0     # invalid sizes -> 0


def test_argument_errors_without_gpu(L):
    assert L.ts_sample_params(0, 0, 4, None) == -2            # TS_ENULL before any CUDA call
    assert b"NULL" in L.ts_last_error()
    out = binding._Out(None, None)
    assert L.ts_render(ctypes.c_void_p(16), 4, 44100, 1.0, out) == -2
    bad = binding.ts_default_nebula()
    bad["curve"][3] = 0.0
    with pytest.raises(binding.TsynthError):
        binding.ts_set_nebula(bad)
    binding.ts_set_nebula(None)


def test_workloads_are_the_baseline_configs():
    w = W.WORKLOADS
    assert [(w[k].B, w[k].sr, w[k].seconds) for k in ("C1", "C2", "C3", "C4", "C5")] == \
        [(4, 44100, 1.0), (128, 44100, 4.0), (1024, 44100, 4.0), (64, 48000, 30.0), (4096, 44100, 4.0)]
    assert w["C2"].N == 176400 and w["C4"].N == 1440000 and w["C3"].batches == 100


def test_c5_edit_lands_in_top_decile_of_human_range():
    wl = W.WORKLOADS["C5"]
    u, _ = O.sample_params(0, 0, 64)
    e = W.edit_u(u, wl)
    neb = W.apply_nebula(O.default_nebula(), wl)
    assert neb["hi"][1] == 4.0
    for b in range(64):
        h = O.map_all(e[b], neb)
        assert h[32] >= 18.0 - 1e-9 and h[40] >= 18.0 - 1e-9           # LFO rate: top 10 % of 0..20 Hz
        assert h[69] >= 76.8 - 1e-9 and h[72] >= 76.8 - 1e-9           # depth: top 10 % of -96..96 st
        if b % 2:
            assert e[b, 76] == 1.0 and e[b, 75] <= 0.25 and e[b, 77] <= 0.25
    assert np.array_equal(W.edit_u(u, wl), e)                          # deterministic, input untouched
    assert np.array_equal(W.edit_u(u, W.WORKLOADS["C2"]), u)


def test_c4_edit_holds_the_note_at_the_top():
    wl = W.WORKLOADS["C4"]
    u, _ = O.sample_params(0, 0, 4)
    h = O.map_all(W.edit_u(u, wl)[0], W.apply_nebula(O.default_nebula(), wl))
    assert h[0] == 127.0 and h[1] == 30.0 and h[69] == 96.0 and h[72] == 96.0


def test_corpus_is_test_matches_oracle_host_only():
    import oracle as O
    import paper_2104_12922_b200 as ts
    for g in list(range(0, 30000, 257)) + [9216, 10239, 10240, 2**40 * 10240 + 9 * 1024 + 5, 2**63 + 9 * 1024]:
        assert ts.ts_corpus_is_test(g) == O.corpus_is_test(g), g
