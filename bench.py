#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path (sampler -> setup -> control -> audio) on synthetic workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--repeats R] [--workload C2] [--impl ours|reference]

A step = one batch of the workload (BASELINE.json configs[1] = C2 by default: 128 voices x 4 s at 44.1 kHz) through the
streaming call ts_corpus_render, batch index = the step number (streaming corpus generation).  The K-step timed
region is repeated R times (each bracketed by a barrier and a device synchronisation); `value` is the median region.
Prints ONE JSON line (rank 0).  `--gpus N` outside torchrun starts the N ranks itself.  `--impl reference` times the CPU
oracle on the host cores instead.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "audio samples/sec"
UNIT = "samples/s"
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def audio_kernel_source_sha() -> str:
    """What a stored per-launch counter of the audio kernel is tied to: the kernel's source file."""
    with open(os.path.join(ROOT, "paper_2104_12922_b200", "csrc", "ts_audio.cu"), "rb") as f:
        return hashlib.sha256(f.read()).hexdigest()[:16]


def ncu_value(name: str, workload: str):
    """A per-launch counter of the audio kernel from the committed summary of the latest `ncu --set full` capture
    (profiles/<name>.csv: workload,value,sha of csrc/ts_audio.cu at the capture), if any -> (value, stale).  stale: the kernel
    source has changed since the capture (or the row carries no sha).  audio_kernel_traffic = dram__bytes_read.sum +
    dram__bytes_write.sum."""
    p = os.path.join(ROOT, "profiles", name + ".csv")
    try:
        with open(p) as f:
            for ln in f:
                cols = ln.strip().split(",")
                if cols[0] == workload:
                    return float(cols[1]), not (len(cols) > 2 and cols[2] == audio_kernel_source_sha())
    except Exception:
        pass
    return None, None


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


class ClockSampler:
    """Polls NVML (the library behind nvidia-smi) for SM clock and throttle reasons while a region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _poll(self):
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def __enter__(self):
        if self.nv:
            self._thr = threading.Thread(target=self._poll, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr:
            self._thr.join()

    def summary(self):
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_samples_per_s(wl, voices: int, repeats: int, threads: int):
    import numpy as np
    import oracle as O
    from paper_2104_12922_b200 import workloads as W
    O.build()
    neb = W.apply_nebula(O.default_nebula(), wl)
    u, nk = O.sample_params(wl.seed, 0, wl.B)
    u = W.edit_u(u, wl)[:voices]
    nk = nk[:voices]
    O.render_batch(u[:1], nk[:1], wl.sr, min(wl.N, 4410), neb, threads=1)   # load the library
    t0 = time.perf_counter()
    for _ in range(repeats):
        O.render_batch(u, nk, wl.sr, wl.N, neb, threads=threads, dtype=np.float32)
    dt = time.perf_counter() - t0
    return repeats * voices * wl.N / dt, dt


def run_reference(args, wl):
    """Base contract's reference arm for this tier: the oracle, as it stands, on the host cores."""
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    voices = min(wl.B, 2 * cores)                 # bounded sample per step
    for _ in range(args.warmup):
        oracle_samples_per_s(wl, min(voices, cores), 1, cores)
    t0 = time.perf_counter()
    total = 0
    for _ in range(args.steps):
        oracle_samples_per_s(wl, voices, 1, cores)
        total += voices * wl.N
    dt = time.perf_counter() - t0
    value = total / dt
    sample = f"{voices} of {wl.B} voices x {wl.seconds} s per step, {cores} threads"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{wl.name}: B={wl.B} x {wl.seconds} s @ {wl.sr} Hz (oracle on a bounded sample: {sample})"},
        "x_real_time": value / wl.sr,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "cpu_model": cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def device_records(ts, W, wl, dev):
    """The workload's parameter records on the device: the GPU's own draw, host-side edits of u (inputs, not method
    arithmetic: workloads.py) applied once and uploaded."""
    import torch
    rec = ts.ts_sample_params(wl.seed, 0, wl.B, device=dev)
    if wl.edit == "none":
        return rec
    h = rec.cpu().numpy()
    h[:, :78] = W.edit_u(h[:, :78], wl, 0)
    return torch.from_numpy(h).to(dev)


_ALU_PEAK = {}
MUFU_PER_RUN = 100   # MUFU warp instructions per 20-sample run (profiles/r02_audio_sass_histogram.txt, whole-cycle variant)
SM_COUNT = 148


def alu_peak(ts):
    """Audible samples/s the SM pipes sustain on the audio kernel's own sample loop (ts_time_alu_bound: the same device
    function, no memory, no CTA turnover, 8 warps per sub-partition), measured once per process: MUFU.SIN variant of the
    square/saw sine (taken by 89 % of the voices) and polynomial variant."""
    if not _ALU_PEAK:
        _ALU_PEAK["fastsin"] = max(ts.ts_time_alu_bound(True, 64) for _ in range(3))
        _ALU_PEAK["poly"] = max(ts.ts_time_alu_bound(False, 64) for _ in range(3))
    return _ALU_PEAK


def kernel_roofline(ts, wl, rec, audio_ring, sm_hz, reps):
    """Per-kernel device times (CUDA events around `reps` back-to-back launches of each, ts_time_kernels), the active
    (non-silent) sample fraction, and the two bounds of the audio kernel."""
    B, sr, seconds, N = wl.B, wl.sr, wl.seconds, wl.N
    ctl, aud = ts.ts_time_kernels(rec, sr, seconds, audio_ring, reps)
    ts.ts_set_timing(True)
    ts.ts_render(rec, sr, seconds, out=audio_ring[0])
    ts.ts_sync()                                   # the active-sample count is valid after ts_sync
    stats = ts.ts_last_stats()
    ts.ts_set_timing(False)
    active = stats["active_samples"] / float(B * N)
    peak, peak_src = measured_peak()
    out_bytes = B * N * 4
    achieved = out_bytes / (aud * 1e-3) / 1e9
    peaks = alu_peak(ts)
    own_pk = peaks["fastsin"]                                               # the higher of the two: a conservative fraction
    aud_ach = stats["active_samples"] / (aud * 1e-3)                        # audible samples/s of this launch
    pipes = ts.ts_time_pipes()
    # The hardware bound of the audible samples: the XU (MUFU) pipe.  A warp renders a 20-sample run of its 32 lanes = 640
    # samples with MUFU_PER_RUN MUFU warp instructions (SASS histogram, profiles/r02_audio_sass_histogram.txt: SIN for VCO 1,
    # SIN + COS for the square/saw, EX2 + RCP for the tanh, per sample, in the whole-cycle variant 89 % of the voices take);
    # ts_time_pipes measures what one MUFU costs a sub-partition (8.0 cycles per warp instruction: 4 lanes per clock).
    xu_peak = 640.0 / (MUFU_PER_RUN * pipes["MUFU.EX2"]) * 4 * SM_COUNT * sm_hz
    t_hbm, t_xu = out_bytes / (peak * 1e9), stats["active_samples"] / xu_peak
    return {"audio_kernel_ms": aud, "control_kernel_ms": ctl, "achieved_gbs": achieved, "frac": achieved / peak,
            "peak": peak, "peak_source": peak_src, "active_sample_fraction": active, "chunks": stats["chunks"],
            "xu_bound": {"bound": "alu", "pipe": "XU (MUFU)", "achieved": aud_ach, "peak": xu_peak, "unit": "audible samples/s",
                         "frac": aud_ach / xu_peak,
                         "derivation": f"640 samples per warp-run / ({MUFU_PER_RUN} MUFU per run x {pipes['MUFU.EX2']:.2f} cycles per MUFU warp "
                                       f"instruction per sub-partition, measured in this run by ts_time_pipes) x 4 sub-partitions x "
                                       f"{SM_COUNT} SMs x {sm_hz / 1e6:.0f} MHz (SM clock sampled under load)"},
            "governing_bound": "xu" if t_xu > t_hbm else "hbm",
            "governing_frac": max(t_hbm, t_xu) / (aud * 1e-3),
            "governing_frac_note": "max(algorithmic bytes / HBM peak, audible samples / XU bound) / kernel duration: the launch against "
                                   "whichever hardware bound is the longer for this workload",
            "own_loop_rate": {"what": "NOT a roofline: audible samples/s of the kernel's own sample loop timed alone (ts_time_alu_bound: "
                              "same device function, no memory, no CTA turnover, 8 warps per sub-partition; MUFU.SIN variant).  It moves "
                              "with the code, so `frac` only says how much of the launch is spent outside the loop (headers, table loads, "
                              "hops, stores, CTA turnover)", "achieved": aud_ach, "rate": own_pk,
                              "rate_polynomial_sine_variant": peaks["poly"], "unit": "audible samples/s", "frac": aud_ach / own_pk,
                              "cycles_per_warp_instruction_per_subpartition": pipes}}


def measure_config(ts, W, torch, name, dev, sm_hz):
    """One extra workload (C1, C3, C4, C5) on rank 0: whole-path step time (median and best of 5 regions) and the audio
    kernel's roofline numbers.  C3 streams consecutive batch indices through ts_corpus_render (sampler included); C4 / C5
    render the same edited records repeatedly through ts_render (setup + control + audio; the 2.5 us sampler is not in
    their step)."""
    wl = W.WORKLOADS[name]
    B, sr, seconds, N = wl.B, wl.sr, wl.seconds, wl.N
    ts.ts_set_nebula(W.apply_nebula(ts.ts_default_nebula(), wl))
    out_bytes = B * N * 4
    nbuf = min(256, max(2, -(-(160 << 20) // out_bytes) + 1))
    lanes = ts.ts_streaming_lanes()
    nbuf += -nbuf % lanes     # a ring that is a multiple of the streaming lanes keeps every slot on one audio stream (no cross-stream events)
    audio_ring = torch.empty((nbuf, B, N), dtype=torch.float32, device=dev)
    rec = device_records(ts, W, wl, dev)
    steps = max(3, min(200, int(0.02 / (out_bytes / 2.0e12))))       # ~20 ms of device time per region
    regions = []
    if wl.edit == "none":
        params_ring = torch.empty((nbuf, B, 80), dtype=torch.float32, device=dev)
        ts.ts_corpus_render(wl.seed, 0, 3, sr, seconds, params_ring, audio_ring)
        how = "ts_corpus_render over consecutive batch indices (sampler + setup + control + audio)"
    else:
        for k in range(3):
            ts.ts_render(rec, sr, seconds, out=audio_ring[k % nbuf])
        how = "ts_render on the edited records (setup + control + audio)"
    torch.cuda.synchronize()
    for r in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        if wl.edit == "none":
            ts.ts_corpus_render(wl.seed, 3 + r * steps, steps, sr, seconds, params_ring, audio_ring)
        else:
            for k in range(steps):
                ts.ts_render(rec, sr, seconds, out=audio_ring[k % nbuf])
        e1.record()
        torch.cuda.synchronize()
        regions.append(e0.elapsed_time(e1) / steps)
    med, best = statistics.median(regions), min(regions)
    roof = kernel_roofline(ts, wl, rec, audio_ring, sm_hz, 20 if out_bytes < (200 << 20) else 4)
    sps = B * N / (med * 1e-3)
    res = {"workload": f"{name}: B={B} voices x {seconds} s @ {sr} Hz", "how": how, "steps_per_region": steps, "regions": 5,
           "ms_per_step": med, "ms_per_step_best": best, "samples_per_s": sps, "x_real_time": sps / sr,
           "audible_samples_per_s": sps * roof["active_sample_fraction"],
           "audio_kernel_ms": roof["audio_kernel_ms"], "control_kernel_ms": roof["control_kernel_ms"], "frac": roof["frac"],
           "xu_frac": roof["xu_bound"]["frac"], "governing_bound": roof["governing_bound"], "governing_frac": roof["governing_frac"],
           "own_loop_frac": roof["own_loop_rate"]["frac"], "active_sample_fraction": roof["active_sample_fraction"],
           "step_over_audio_kernel": med / roof["audio_kernel_ms"], "voice_chunks_per_launch": roof["chunks"]}
    del audio_ring
    torch.cuda.empty_cache()
    return res


def run_ours(args, wl):
    import torch
    import paper_2104_12922_b200 as ts
    from paper_2104_12922_b200 import build, shard, workloads as W
    build.build()
    ts.use_measure_build()   # libtsynth_measure.so: the product's sources + the ts_time_* aids (include/tsynth_measure.h)
    rank, local_rank, world = shard.init("nccl")
    if world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE is {world}")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    B, sr, seconds, N = wl.B, wl.sr, wl.seconds, wl.N
    if wl.edit != "none":
        raise SystemExit("the headline workload streams batch indices (C1, C2, C3); C4 / C5 are reported under `configs`")
    ts.ts_set_nebula(W.apply_nebula(ts.ts_default_nebula(), wl))

    # rotating output buffers: together larger than the 126 MB L2, so no step rewrites lines still cached
    out_bytes = B * N * 4
    nbuf = min(256, max(2, -(-(160 << 20) // out_bytes) + 1))
    lanes = ts.ts_streaming_lanes()
    nbuf += -nbuf % lanes     # a ring that is a multiple of the streaming lanes keeps every slot on one audio stream (no cross-stream events)
    audio_ring = torch.empty((nbuf, B, N), dtype=torch.float32, device=dev)
    params_ring = torch.empty((nbuf, B, 80), dtype=torch.float32, device=dev)

    # ---- the timed regions: K consecutive batch indices of this rank's contiguous range through the streaming call
    # (sampler + setup + control + audio per batch, consecutive batches on the internal streaming lanes), R times
    K, Wm, R = args.steps, args.warmup, args.repeats
    per_rank = Wm + K * R
    first, _count = shard.batch_range(rank, world, per_rank)
    ts.ts_corpus_render(wl.seed, first, Wm, sr, seconds, params_ring, audio_ring)
    torch.cuda.synchronize()
    regions = []
    launches = 0
    with ClockSampler(local_rank) as clk:
        for r in range(R):
            shard.barrier()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ts.ts_corpus_render(wl.seed, first + Wm + r * K, K, sr, seconds, params_ring, audio_ring)
            e1.record()
            torch.cuda.synchronize()
            shard.barrier()
            regions.append(shard.max_over_ranks(e0.elapsed_time(e1), dev))
            launches = ts.ts_last_stats()["launches"]
    ms = statistics.median(regions)
    total_samples = float(B) * N * K * world
    value = total_samples / (ms * 1e-3)
    clocks = clk.summary()
    sm_hz = 1e6 * float(clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965)

    # ---- roofline of the dominant kernel (audio): algorithmic bytes = 4 B per output sample
    rec = device_records(ts, W, wl, dev)
    roof = kernel_roofline(ts, wl, rec, audio_ring, sm_hz, 50)
    try:
        two_ms = min(ts.ts_time_audio_lanes(rec, sr, seconds, audio_ring, 50) for _ in range(3))
    except ts.TsynthError:  # the batch needs several voice chunks (C3): the overlapped-launch figure is a one-chunk measurement
        two_ms = None
    fill_ms = ts.ts_time_fill(audio_ring, 5)
    fill_gbs = audio_ring.numel() * 4 / (fill_ms * 1e-3) / 1e9
    traffic, traffic_stale = ncu_value("audio_kernel_traffic", wl.name)
    roofline = {"bound": "hbm", "kernel": "ts_audio_kernel<0, TAIL, F32>", "achieved": roof["achieved_gbs"], "peak": roof["peak"],
                "unit": "GB/s", "frac": roof["frac"],
                "achieved_is": "ALGORITHMIC bytes per launch (4 B per output sample) / the kernel's launch duration measured in this run; "
                               "not measured DRAM traffic (that is `traffic`)",
                "traffic": traffic, "traffic_stale": traffic_stale,
                "traffic_source": "stored value: dram__bytes_read.sum + dram__bytes_write.sum of one launch in the committed "
                                  "`ncu --set full` capture (profiles/audio_kernel_traffic.csv, tied to the sha of csrc/ts_audio.cu: "
                                  "traffic_stale = the kernel source has changed since), not measured in this run; it is "
                                  "below the algorithmic bytes because the 126 MB L2 still holds the end of a single launch's writes",
                "xu_bound": roof["xu_bound"], "frac_xu": roof["xu_bound"]["frac"],
                "governing_bound": roof["governing_bound"], "governing_frac": roof["governing_frac"],
                "governing_frac_note": roof["governing_frac_note"],
                "peak_source": roof["peak_source"], "algorithmic_bytes_per_launch": out_bytes,
                "audio_kernel_ms": roof["audio_kernel_ms"], "control_kernel_ms": roof["control_kernel_ms"],
                "timing": "CUDA events around 50 back-to-back launches of each kernel (ts_time_kernels); control = setup + control",
                "audio_kernel_ms_two_streams": two_ms,
                "frac_two_streams": out_bytes / (two_ms * 1e-3) / 1e9 / roof["peak"] if two_ms else None,
                "own_loop_frac_two_streams": roof["active_sample_fraction"] * B * N / (two_ms * 1e-3) / roof["own_loop_rate"]["rate"] if two_ms else None,
                "audio_kernel_ms_two_streams_note": "interval / launches with the launches rotating over the audio streams of the streaming lanes, as "
                                                    "the streaming calls issue them: an inverse throughput (the ramp and drain of a launch are "
                                                    "covered by the other stream) of AUDIO-ONLY launches with no control kernels competing for the SMs, not the "
                                                    "launch duration `frac` is computed from and not what the pipeline reaches: that is "
                                                    "whole_step_frac_of_write_roofline",
                "store_only_fill_gbs": fill_gbs,
                "store_only_fill": f"{audio_ring.numel() * 4 >> 20} MiB of 128-bit zero stores, 5 launches (ts_time_fill): what a pure "
                                   "store stream reaches, beside the copy peak above",
                "active_sample_fraction": roof["active_sample_fraction"], "own_loop_rate": roof["own_loop_rate"],
                "note": "audible samples are bound by the SM pipes (XU: 5 MUFU per sample; FMA-heavy: Philox IMAD.WIDE + packed fp32; ~46 "
                        "SASS instructions each), silent tails are pure stores written asynchronously by the audible CTAs; the two "
                        "hardware bounds are `frac` (HBM writes) and `frac_xu` (MUFU pipe), `governing_frac` the launch against the longer",
                "whole_step_frac_of_write_roofline": (4.0 * value / world / 1e9) / roof["peak"]}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 (audio) + f64 / Q0.64 (control and phase chain)", "data": "synthetic",
            "config": {"workload": f"{wl.name}: B={B} voices x {seconds} s @ {sr} Hz per GPU per step, seed 0, consecutive batch "
                                   "indices through ts_corpus_render (sampler + setup + control + audio per batch)",
                       "l2": f"{nbuf} rotating output buffers of {out_bytes >> 20} MiB (> 126 MB L2 together)",
                       "partition": f"rank r renders the contiguous batch-index range [r*{per_rank}, (r+1)*{per_rank})"},
            "timing": {"repeats": R, "ms_per_step_median": ms / K, "ms_per_step_best": min(regions) / K,
                       "ms_per_step_all": [x / K for x in regions],
                       "how": "each repeat = exactly K steps between two CUDA events, barrier + synchronize on both sides, max over ranks"},
            "x_real_time": value / sr, "audible_samples_per_s": value * roof["active_sample_fraction"],
            "step_over_audio_kernel": (ms / K) / roof["audio_kernel_ms"],
            "clocks": clocks, "gpu_launches": int(launches) * world,
            "roofline": roofline,
            "paper_context": "714e6 samples/s on one V100 (P:L23); other hardware, context only"}

    # ---- end to end through the public host-buffer call: sample + render + D2H of audio and records, fp32 and fp16
    if rank == 0 or world > 1:
        n_e2e = max(3, min(K, 10))
        first_e2e, _ = shard.batch_range(rank, world, n_e2e + 1)
        for key, fmt, dt, es in (("e2e", ts.TS_F32, torch.float32, 4), ("e2e_f16", ts.TS_F16, torch.float16, 2)):
            host = torch.empty((B, N), dtype=dt, pin_memory=True)
            hostp = torch.empty((B, 80), dtype=torch.float32, pin_memory=True)
            ts.ts_render_host_fmt(wl.seed, first_e2e, B, sr, seconds, fmt, host, hostp)
            shard.barrier()
            t0 = time.perf_counter()
            for i in range(n_e2e):
                ts.ts_render_host_fmt(wl.seed, first_e2e + 1 + i, B, sr, seconds, fmt, host, hostp)
            dt_s = shard.max_over_ranks(time.perf_counter() - t0, dev)
            line[key] = {"value": float(B) * N * n_e2e * world / dt_s, "unit": UNIT, "h2d_bytes_per_step": 0,
                         "d2h_bytes_per_step": B * N * es + B * 320, "steps": n_e2e,
                         "note": "inputs are (seed, batch index) scalars: nothing to copy host->device; PCIe-bound on the audio copy"}

    if rank == 0 and world == 1:
        # ---- the other configs (BASELINE.json configs[0], [2..4]) beside the headline, so that it is not a memset number
        if not args.no_configs:
            line["configs"] = {name: measure_config(ts, W, torch, name, dev, sm_hz) for name in ("C1", "C3", "C4", "C5") if name != wl.name}
            ts.ts_set_nebula(W.apply_nebula(ts.ts_default_nebula(), wl))
        # ---- control-rate call on its own, MMD arithmetic
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ctl_out = ts.ts_render_controls(rec, sr, seconds)
        torch.cuda.synchronize()
        e0.record()
        lib = ts.lib()
        import ctypes as C
        for _ in range(20):
            lib.ts_render_controls(C.c_void_p(rec.data_ptr()), B, sr, float(seconds), C.c_void_p(ctl_out.data_ptr()))
        e1.record()
        torch.cuda.synchronize()
        line["controls_only"] = {"ms_per_call": e0.elapsed_time(e1) / 20, "what": f"ts_render_controls on {wl.name}: {B} voices x "
                                 f"{ctl_out.shape[2]} ticks x 5 rows fp64 (setup + control kernel without the oscillator stage)"}
        n, d = 1000, 512
        g = torch.Generator(device=dev).manual_seed(0)
        X = torch.randn((n, d), device=dev, generator=g)
        Y = 0.7 * torch.randn((n, d), device=dev, generator=g) + 0.3
        mmd = {}
        for form in ("auto", "pairwise", "sorted"):
            ts.ts_mmd_l1(X, Y, form=form)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(20):
                ts.ts_mmd_l1(X, Y, form=form)
            e1.record()
            torch.cuda.synchronize()
            mmd[form] = e0.elapsed_time(e1) / 20
        T = -(-n // 64)
        pair_comps = (T * T + T * (T + 1)) * 64 * 64 * d                 # (pair, component) items computed, padded tiles included
        alu_s = 2.0 * pair_comps / (148 * 128 * sm_hz)                    # 2 FADD-class thread instructions per item
        # the sorted form (the one ts_mmd_l1 runs at this n): a bitonic network of M = 2^L keys per component has (M / 2) L (L + 1) / 2
        # compare-exchanges; one 64-bit compare-exchange is ~11 integer instructions (profiles/r02_final.md) on the half-rate
        # integer pipe, whose cost per warp instruction per sub-partition is measured in this run (ts_time_pipes: LOP3)
        M = 512
        while M < 2 * n:
            M *= 2
        Lg = M.bit_length() - 1
        cmpx = d * (M // 2) * Lg * (Lg + 1) // 2
        int_cycles = roof["own_loop_rate"]["cycles_per_warp_instruction_per_subpartition"]["LOP3"]
        sort_s = (cmpx / 32.0) * 11.0 * int_cycles / (4 * SM_COUNT) / sm_hz
        line["mmd_l1"] = {"ms_per_call": mmd["auto"], "ms_pairwise_form": mmd["pairwise"], "ms_sorted_form": mmd["sorted"],
                          "n": n, "d": d, "bound": "alu", "unit": "s", "peak_s": alu_s, "frac": alu_s / (mmd["pairwise"] * 1e-3),
                          "sorted_form": {"bound": "alu", "pipe": "integer (half rate)", "peak_s": sort_s, "frac": sort_s / (mmd["sorted"] * 1e-3),
                                          "derivation": f"{cmpx} compare-exchanges of 64-bit keys ({d} components x {M // 2} x {Lg * (Lg + 1) // 2} "
                                                        f"network levels) / 32 lanes x ~11 integer instructions x {int_cycles:.2f} cycles per warp "
                                                        f"instruction per sub-partition (measured) / {4 * SM_COUNT} sub-partitions / SM clock; the "
                                                        "strided loads, the 128-bit scan and the reductions (a quarter of the kernel's instructions) "
                                                        "are not in the bound"},
                          "what": "Eq. 2 with the l1 core distance (P:L230).  ts_mmd_l1 runs the faster of two forms: pairwise "
                                  "(O(d n^2); the top-level `bound` / `frac` are this form's: 2 FADD-class instructions per (pair, component) at 148 SMs "
                                  "x 128 fp32 lanes per clock) and sorted (`sorted_form` carries its own bound: (O(d n log^2 n): one bitonic sort of the 2n values of every "
                                  "component in shared memory, exact integer sums)); embeddings (4 MB) are L2-resident"}
        # ---- a nebula sweep in the shape of the paper's tuning runs (256 sounds per candidate table)
        import numpy as np
        nt, Bn = 24, 256
        rng = np.random.default_rng(0)
        tabs = np.stack([ts.ts_default_nebula() for _ in range(nt)])
        for t in tabs:
            t["curve"] = np.exp(rng.uniform(np.log(0.1), np.log(10.0), t.shape[0]))   # log-uniform in [0.1, 10]
        lanes = ts.ts_streaming_lanes()
        prn = torch.empty((lanes, Bn, 80), dtype=torch.float32, device=dev)
        arn = torch.empty((lanes, Bn, N), dtype=torch.float32, device=dev)
        ts.ts_corpus_render_nebulae(wl.seed, 0, sr, seconds, ts.TS_F32, tabs, prn, arn)
        torch.cuda.synchronize()
        e0.record()
        ts.ts_corpus_render_nebulae(wl.seed, nt, sr, seconds, ts.TS_F32, tabs, prn, arn)
        e1.record()
        torch.cuda.synchronize()
        sweep_ms = e0.elapsed_time(e1)
        line["nebula_sweep"] = {"ms_per_table": sweep_ms / nt, "samples_per_s": nt * Bn * N / (sweep_ms * 1e-3), "tables": nt,
                                "voices_per_table": Bn, "what": "ts_corpus_render_nebulae: one candidate table (curves log-uniform in "
                                "[0.1, 10], P:L270) per batch of 256 voices x 4 s, table upload included"}
        del prn, arn
        if not args.no_cpu_baseline:
            cores = os.cpu_count() or 1
            voices = min(wl.B, 128)
            _v, dt1 = oracle_samples_per_s(wl, voices, 1, cores)
            repeats = max(2, min(400, int(12.0 / max(dt1, 1e-3))))           # ~12 s of wall clock on all cores
            v, dt = oracle_samples_per_s(wl, voices, repeats, cores)
            v1, dts = oracle_samples_per_s(wl, 8, 2, 1)                       # and one thread: 8 voices twice
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"first {voices} voices of the batch x {seconds} s, {repeats} repeats, "
                                              f"{dt:.1f} s wall on {cores} threads",
                                    "one_thread": {"value": v1, "unit": UNIT, "sample": f"8 voices x {seconds} s twice, {dts:.1f} s"},
                                    "x_real_time": v / sr, "cpu_model": cpu_model()}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--repeats", type=int, default=21, help="timed regions of exactly --steps steps; value = the median one")
    ap.add_argument("--workload", default="C2", choices=["C1", "C2", "C3"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the C1 / C3 / C4 / C5 entries of the line")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    args.repeats = max(args.repeats, 1)
    from paper_2104_12922_b200 import shard, workloads as W
    wl = W.WORKLOADS[args.workload]
    if args.impl == "reference":
        run_reference(args, wl)
        return
    if args.gpus > 1 and not shard.under_torchrun():
        # `python bench.py --gpus N` without a torchrun environment: start the N ranks ourselves
        sys.exit(shard.respawn_under_torchrun(args.gpus, os.path.abspath(__file__), sys.argv[1:]))
    run_ours(args, wl)


if __name__ == "__main__":
    main()
