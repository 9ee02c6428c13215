"""Seeded, counter-based synthetic uint8 filterbank (test/bench fixture; DATA only).

Recipe (SURVEY.md 8(d) "Generator rule", BASELINE.json configs): every sample is
`clip(round(N(128, 16^2)), 0, 255)`; dispersed pulses of a given DM, start sample, width
and amplitude are then added with saturation at 255.  The paper tuned on "uniformly
distributed noise with injected single pulse signal"; BASELINE.json
replaces that with Gaussian noise -- the configs bind.

Counter-based: sample (c, t) is a pure function of (seed, c, t // 4): one 64-bit mix gives
four 16-bit uniforms, each mapped through a 65536-entry inverse-CDF table of the rounded
and clipped Gaussian (probabilities quantised to 2^-16).  No stream state, so any part of
the array can be generated in any order and chunking never changes the bytes.

This module is shared by the oracle tests and by the CUDA tests/bench.  It implements none
of the search method (no dedispersion sum, no integration, no S/N).  The only physics in
it is the *signal model* of an injected pulse: the cold-plasma arrival-time law
t(f) = t0 + K*DM*(f^-2 - f_ref^-2), which is what makes a dispersed pulse a dispersed pulse.
"""
from __future__ import annotations

import math
from typing import List, Sequence, Tuple

import numpy as np

from .configs import Pulse, SearchConfig

K_DM = 4.148808e3  # s MHz^2 pc^-1 cm^3 (BASELINE.json north_star)

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wraps mod 2^64)."""
    x = x.copy()
    with np.errstate(over="ignore"):
        x ^= x >> np.uint64(30)
        x *= np.uint64(0xBF58476D1CE4E5B9)
        x ^= x >> np.uint64(27)
        x *= np.uint64(0x94D049BB133111EB)
        x ^= x >> np.uint64(31)
    return x


def mix64_scalar(x: int) -> int:
    x &= 0xFFFFFFFFFFFFFFFF
    x ^= x >> 30
    x = (x * 0xBF58476D1CE4E5B9) & 0xFFFFFFFFFFFFFFFF
    x ^= x >> 27
    x = (x * 0x94D049BB133111EB) & 0xFFFFFFFFFFFFFFFF
    x ^= x >> 31
    return x


_TABLE = None


def gaussian_u8_table(mean: float = 128.0, sd: float = 16.0) -> np.ndarray:
    """table[u] for a 16-bit uniform u: the value v in 0..255 whose rounded-and-clipped
    Gaussian CDF interval contains (u + 0.5) / 65536."""
    global _TABLE
    if _TABLE is not None and (mean, sd) == (128.0, 16.0):
        return _TABLE
    cum = np.empty(256, dtype=np.float64)
    for v in range(255):
        z = (v + 0.5 - mean) / sd
        cum[v] = 0.5 * (1.0 + math.erf(z / math.sqrt(2.0)))
    cum[255] = 1.0
    u = (np.arange(65536, dtype=np.float64) + 0.5) / 65536.0
    table = np.searchsorted(cum, u, side="right").astype(np.uint8)
    if (mean, sd) == (128.0, 16.0):
        _TABLE = table
    return table


def noise_rows(seed: int, c0: int, c1: int, nsamp: int) -> np.ndarray:
    """uint8 [c1-c0][nsamp] noise for channels c0..c1-1 (counter-based)."""
    table = gaussian_u8_table()
    nq = (nsamp + 3) // 4
    q = np.arange(nq, dtype=np.uint64)
    out = np.empty((c1 - c0, nq * 4), dtype=np.uint8)
    s0 = np.uint64(mix64_scalar(seed * 0x9E3779B97F4A7C15 + 0x1234567))
    for r, c in enumerate(range(c0, c1)):
        with np.errstate(over="ignore"):
            key = _mix64(np.uint64(c + 1) * np.uint64(0xD6E8FEB86659FD93) ^ s0)
            h = _mix64((q + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15) ^ key)
        u16 = h.view(np.uint16).reshape(nq, 4)  # little-endian: 4 x 16-bit per hash
        out[r] = table[u16].reshape(-1)
    return out[:, :nsamp]


def beam_seed(data_seed: int, beam: int) -> int:
    """Seed of the synthetic filterbank of one beam (beam 0 = the config's own seed)."""
    return int(data_seed) + 7919 * int(beam)


def draw_pulses(cfg: SearchConfig) -> List[Pulse]:
    """The config's pulse list: fixed pulses, plus `n_pulses` hash-drawn ones with the DM on
    the trial grid, width in {1,2,4,8,16,32} (restricted to the config's widths), start a
    multiple of the width in [0, nsamp_out - 64), amplitude 5..30."""
    pulses = list(cfg.fixed_pulses)
    wset = [w for w in (1, 2, 4, 8, 16, 32) if w in cfg.widths] or [cfg.widths[0]]
    for p in range(cfg.n_pulses):
        h = [mix64_scalar((cfg.seed << 20) ^ (0xA5A5 + 7919 * p + k)) for k in range(4)]
        dm_idx = h[0] % cfg.ndm
        width = wset[h[1] % len(wset)]
        span = max(1, (cfg.nsamp_out - 64) // width)
        t0 = (h[2] % span) * width
        amp = 5 + h[3] % 26
        pulses.append(Pulse(dm=cfg.dm_first + cfg.dm_step * dm_idx, t0=int(t0),
                            width=int(width), amplitude=int(amp)))
    return pulses


def pulse_track(cfg: SearchConfig, pulse: Pulse) -> np.ndarray:
    """Arrival sample of the pulse's leading edge in every channel (signal model)."""
    f = cfg.chan_freq_mhz()
    f_ref = f.max()
    g = 1.0 / (f * f) - 1.0 / (f_ref * f_ref)
    return pulse.t0 + np.floor(((K_DM * pulse.dm) * g) / cfg.t_samp_s + 0.5).astype(np.int64)


def make_filterbank(cfg: SearchConfig, nsamp_in: int, in_stride: int = None,
                    chunk: int = 64, bits: int = 8) -> Tuple[np.ndarray, List[Pulse]]:
    """uint8 [nchan][in_stride] (time fastest; columns >= nsamp_in are zero padding).
    bits = 16 (INPUT_BITS = 16): uint16 samples whose high byte is the 8-bit recipe (noise and
    pulses) and whose low byte is a second noise stream of the same recipe (seed + 0x10001), zero in the padding."""
    if in_stride is None:
        in_stride = nsamp_in
    assert in_stride >= nsamp_in and bits in (8, 16)
    if bits == 16:
        hi, pulses = make_filterbank(cfg, nsamp_in, in_stride, chunk)
        X16 = hi.astype(np.uint16) << np.uint16(8)
        lo_seed = cfg.seed + 0x10001
        for c0 in range(0, cfg.nchan, chunk):
            c1 = min(cfg.nchan, c0 + chunk)
            X16[c0:c1, :nsamp_in] |= noise_rows(lo_seed, c0, c1, nsamp_in).astype(np.uint16)
        return X16, pulses
    X = np.zeros((cfg.nchan, in_stride), dtype=np.uint8)
    for c0 in range(0, cfg.nchan, chunk):
        c1 = min(cfg.nchan, c0 + chunk)
        X[c0:c1, :nsamp_in] = noise_rows(cfg.seed, c0, c1, nsamp_in)
    pulses = draw_pulses(cfg)
    for p in pulses:
        track = pulse_track(cfg, p)
        for c in range(cfg.nchan):
            a = int(track[c])
            b = min(nsamp_in, a + p.width)
            if a < nsamp_in and b > a:
                seg = X[c, a:b].astype(np.int32) + p.amplitude
                X[c, a:b] = np.minimum(seg, 255).astype(np.uint8)
    return X, pulses
