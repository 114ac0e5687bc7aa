"""Seeded synthetic workloads C1..C5 (BASELINE.json configs[0..4]).

Serves both the CUDA path and the oracle's tests.  Holds NONE of the method's arithmetic: it names
sizes, nebula range overrides, and edits of the normalised parameter matrix u[B,78] (which each side
draws with its own Philox sampler).  All constants below are stated in DESIGN.md.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

NPARAM = 78
# normalised value above which the default nebula's curve lands in the top 10 % of the human range:
#   lfo frequency (idx 32, 40): lo + (hi-lo) u^4      >= hi - 0.1 (hi-lo)  <=>  u >= 0.9^(1/4)
#   vco mod depth (idx 69, 72): centre + half |2u-1|^5 >= hi - 0.1 (hi-lo)  <=>  u >= (1 + 0.8^(1/5)) / 2
U_TOP10_LFO_FREQ = 0.9740037464252967
U_TOP10_MOD_DEPTH = 0.9781966575012527


@dataclass(frozen=True)
class Workload:
    name: str
    B: int
    sr: int
    seconds: float
    seed: int = 0
    batches: int = 1                    # consecutive batch indices (C3 streams 100)
    nebula_hi: dict = field(default_factory=dict)   # {param index: new `hi`} applied to the default nebula
    edit: str = "none"                  # which edit_u() rule applies

    @property
    def N(self) -> int:
        return int(round(self.sr * self.seconds))


WORKLOADS = {
    "C1": Workload("C1", 4, 44100, 1.0),
    "C2": Workload("C2", 128, 44100, 4.0),
    "C3": Workload("C3", 1024, 44100, 4.0, batches=100),
    "C4": Workload("C4", 64, 48000, 30.0, nebula_hi={1: 30.0}, edit="c4"),
    "C5": Workload("C5", 4096, 44100, 4.0, nebula_hi={1: 4.0}, edit="c5"),
}


def apply_nebula(neb: np.ndarray, wl: Workload) -> np.ndarray:
    """neb: structured array [78] (lo, hi, curve, symmetric) of either side -> copy with wl's overrides."""
    out = neb.copy()
    for idx, hi in wl.nebula_hi.items():
        out["hi"][idx] = hi
    return out


def edit_u(u: np.ndarray, wl: Workload, first_voice: int = 0) -> np.ndarray:
    """u: float32 [B,78] drawn by a sampler -> the matrix both sides render (a copy)."""
    u = np.array(u, dtype=np.float32, copy=True)
    if wl.edit == "c4":
        # MIDI 127, +96 st depth on both VCOs, note held for the whole 30 s (duration.hi = 30)
        u[:, 0] = 1.0
        u[:, 69] = 1.0
        u[:, 72] = 1.0
        u[:, 1] = 1.0
    elif wl.edit == "c5":
        for idx, lo in ((32, U_TOP10_LFO_FREQ), (40, U_TOP10_LFO_FREQ), (69, U_TOP10_MOD_DEPTH), (72, U_TOP10_MOD_DEPTH)):
            u[:, idx] = (np.float64(lo) + (1.0 - np.float64(lo)) * u[:, idx].astype(np.float64)).astype(np.float32)
        odd = ((np.arange(u.shape[0]) + first_voice) % 2) == 1   # square/saw-dominant half
        u[odd, 76] = 1.0
        u[odd, 75] *= np.float32(0.25)
        u[odd, 77] *= np.float32(0.25)
    return u
