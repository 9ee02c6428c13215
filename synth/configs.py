"""Shapes of the five BASELINE.json workloads (no method arithmetic lives here).

`BJ:cfgN` = BASELINE.json `configs[N]`; SURVEY.md section 8(d) table "Synthetic inputs"
fixes the seeds and the frequency convention FRQ.1 (top channel exactly f_hi, channel
spacing (f_hi - f_lo)/nchan, mirroring PAPER.md Table 2).

A `SearchConfig` is pure data: channel frequencies, sampling time, DM grid, widths,
pulse list.  Both the oracle tests and the CUDA tests/bench build their inputs from it.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

BASE_SEED = 1811041650  # data seed = BASE_SEED + config index


@dataclass(frozen=True)
class Pulse:
    dm: float        # pc cm^-3
    t0: int          # first sample at the reference (top) frequency
    width: int       # samples
    amplitude: int   # counts added to every channel


@dataclass(frozen=True)
class SubbandPlan:
    n_subbands: int
    n_coarse: int
    coarse_first: float
    coarse_step: float
    n_fine: int
    fine_step: float


@dataclass(frozen=True)
class SearchConfig:
    name: str
    nchan: int
    f_hi_mhz: float
    f_lo_mhz: float
    t_samp_s: float
    nsamp_out: int
    dm_first: float
    dm_step: float
    ndm: int
    widths: Tuple[int, ...]
    seed: int
    n_pulses: int
    subband: Optional[SubbandPlan] = None
    fixed_pulses: Tuple[Pulse, ...] = field(default_factory=tuple)

    # --- derived, plain data -------------------------------------------------
    def chan_freq_mhz(self) -> np.ndarray:
        """FRQ.1: f[c] = f_hi - c*(f_hi - f_lo)/nchan, c = 0..nchan-1 (descending)."""
        c = np.arange(self.nchan, dtype=np.float64)
        return self.f_hi_mhz - c * ((self.f_hi_mhz - self.f_lo_mhz) / self.nchan)

    def dm_list(self) -> np.ndarray:
        return self.dm_first + self.dm_step * np.arange(self.ndm, dtype=np.float64)


def _pow2(lo: int, hi: int) -> Tuple[int, ...]:
    out, w = [], lo
    while w <= hi:
        out.append(w)
        w *= 2
    return tuple(out)


def tiny() -> SearchConfig:
    """BJ:cfg0 -- oracle finishes in seconds."""
    return SearchConfig(
        name="cfg0_tiny", nchan=64, f_hi_mhz=1550.0, f_lo_mhz=1250.0, t_samp_s=81.92e-6,
        nsamp_out=4096, dm_first=0.0, dm_step=1.0, ndm=32, widths=(1, 2, 4, 8),
        seed=BASE_SEED + 0, n_pulses=0,
        fixed_pulses=(Pulse(dm=17.0, t0=2000, width=4, amplitude=20),))


def apertif_direct() -> SearchConfig:
    """BJ:cfg1 -- Apertif-like direct dedispersion (the bench workload)."""
    return SearchConfig(
        name="cfg1_apertif_direct", nchan=1536, f_hi_mhz=1550.0, f_lo_mhz=1250.0,
        t_samp_s=40.96e-6, nsamp_out=24414, dm_first=0.0, dm_step=0.25, ndm=2048,
        widths=_pow2(1, 256), seed=BASE_SEED + 1, n_pulses=8)


def apertif_subband() -> SearchConfig:
    """BJ:cfg2 -- two-step subband on cfg1's bytes (same seed => identical input)."""
    return SearchConfig(
        name="cfg2_apertif_subband", nchan=1536, f_hi_mhz=1550.0, f_lo_mhz=1250.0,
        t_samp_s=40.96e-6, nsamp_out=24414, dm_first=0.0, dm_step=0.25, ndm=2048,
        widths=_pow2(1, 256), seed=BASE_SEED + 1, n_pulses=8,
        subband=SubbandPlan(n_subbands=32, n_coarse=64, coarse_first=0.0, coarse_step=8.0,
                            n_fine=32, fine_step=0.25))


def ska_mid() -> SearchConfig:
    """BJ:cfg3 -- SKA-Mid-like large search."""
    return SearchConfig(
        name="cfg3_ska_mid", nchan=4096, f_hi_mhz=950.0, f_lo_mhz=650.0, t_samp_s=50e-6,
        nsamp_out=20000, dm_first=0.0, dm_step=0.5, ndm=4096, widths=_pow2(1, 512),
        seed=BASE_SEED + 3, n_pulses=16)


def scaled(base: SearchConfig, *, name: str, nchan: int = None, nsamp_out: int = None,
           ndm: int = None, widths: Tuple[int, ...] = None, n_pulses: int = None,
           subband: Optional[SubbandPlan] = None, seed: int = None) -> SearchConfig:
    """A reduced copy of a config (same band, sampling and value recipe) for tests whose
    oracle leg must finish in seconds."""
    import dataclasses
    kw = {"name": name}
    if nchan is not None: kw["nchan"] = nchan
    if nsamp_out is not None: kw["nsamp_out"] = nsamp_out
    if ndm is not None: kw["ndm"] = ndm
    if widths is not None: kw["widths"] = widths
    if n_pulses is not None: kw["n_pulses"] = n_pulses
    if seed is not None: kw["seed"] = seed
    kw["subband"] = subband
    return dataclasses.replace(base, **kw)


ALL = {"cfg0": tiny, "cfg1": apertif_direct, "cfg2": apertif_subband, "cfg3": ska_mid}
