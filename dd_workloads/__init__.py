"""Seeded synthetic filterbank inputs for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests, cpu_baseline) and the CUDA path
(tests, bench) and therefore holds NONE of the method's arithmetic: no delay
formula, no dedispersion sum, no unpacking.  Where an input needs a dispersion
track (the injected pulses of configs 1 and 3) the caller passes the delay rows
in (`tracks`); this module never computes a delay.

Generator: counter based, so that (i) a multi-GB input can be produced directly
in HBM by the same integer code that produces it on the host, and (ii) any single
sample (beam, c, t) can be evaluated on its own, which is what lets the oracle
check sampled outputs of the full-size configs one by one.

    h(seed, beam, c, t) = splitmix64_finalise( (seed + 1000*beam)*G0 + c*G1 + t*G2 )   (mod 2^64)
    uniform 2-bit : h >> 62            uniform 4-bit : h >> 60
    "gauss"       : S = sum of the 8 bytes of h (Irwin-Hall, mean 1020, sigma 209.02)
                    v = clip(128 + round_half_up((S - 1020) * sigma / 209.02), 0, 255)

All arithmetic is 64-bit integer (torch int64 with two's-complement wrap-around),
identical on CPU and CUDA tensors.  The recipe is stated in DESIGN.md §4.

Packing (reading R9 of DESIGN.md): sample t of a row lives in byte (t*nbits)>>3,
bits [(t*nbits)&7, +nbits), LSB first.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional, Sequence

import numpy as np
import torch

BASE_SEED = 12015380  # arXiv id 1201.5380

_G0 = 0x9E3779B97F4A7C15
_G1 = 0xBF58476D1CE4E5B9
_G2 = 0x94D049BB133111EB
_MASK64 = (1 << 64) - 1

# Irwin-Hall(8 bytes): variance 8*(256^2-1)/12 = 43690 -> sigma = 209.0215...
_IH_MEAN = 1020
_IH_SIGMA_X1E4 = 2090215  # sigma * 1e4, integer


def _s64(x: int) -> int:
    """Python int (mod 2^64) -> the int64 with the same bit pattern."""
    x &= _MASK64
    return x - (1 << 64) if x >= (1 << 63) else x


@dataclass(frozen=True)
class Config:
    """One BASELINE.json workload (or a reduced copy of one for parity tests)."""
    name: str
    index: int                 # 1..5, position in BASELINE.json `configs`
    nchans: int
    f_top: float               # MHz, frequency of channel 0
    df: float                  # MHz, channel width (negative: descending)
    dt: float                  # s
    nbits: int                 # 2 | 4 | 8
    nsamps: int                # OUTPUT samples per DM trial
    ndm: int
    dm_max: float              # DM list is d*dm_max/(ndm-1), d = 0..ndm-1 (inclusive end)
    out: str                   # "f32" | "u32" | "u16"
    dist: str                  # "uniform" | "gauss"
    sigma: int = 0             # for "gauss"
    nbeams: int = 1
    npulses: int = 0
    pulse_amp: int = 40
    pulse_dm_index: Optional[int] = None   # config 1: fixed DM trial (DM 50 -> d = 10)
    seed: int = field(default=0)

    @property
    def out_nbits(self) -> int:
        """The dd_execute `out_nbits` code for this config's output type."""
        return {"f32": 32, "u32": -32, "u16": 16}[self.out]

    def dm_list(self) -> np.ndarray:
        """Uniform, end-inclusive DM list in float64 (reading R14)."""
        if self.ndm == 1:
            return np.zeros(1, dtype=np.float64)
        d = np.arange(self.ndm, dtype=np.float64)
        return d * self.dm_max / float(self.ndm - 1)

    def reduced(self, *, nsamps: int, ndm: Optional[int] = None, nbeams: Optional[int] = None,
                nchans: Optional[int] = None, name_suffix: str = "-reduced") -> "Config":
        """A smaller copy with the same band, DM spacing and value distribution.

        `ndm` keeps the DM *step* (so per-trial delay steps stay those of the real
        config) and therefore lowers dm_max; `nchans` keeps f_top and df.
        """
        ndm_new = self.ndm if ndm is None else ndm
        step = self.dm_max / float(self.ndm - 1) if self.ndm > 1 else 0.0
        return replace(self, name=self.name + name_suffix, nsamps=nsamps, ndm=ndm_new,
                       dm_max=step * (ndm_new - 1),
                       nbeams=self.nbeams if nbeams is None else nbeams,
                       nchans=self.nchans if nchans is None else nchans,
                       pulse_dm_index=(None if self.pulse_dm_index is None
                                       else min(self.pulse_dm_index, ndm_new - 1)))


def _cfg(index, **kw) -> Config:
    return Config(index=index, seed=BASE_SEED + index, **kw)


CONFIGS = {
    1: _cfg(1, name="cfg1-tiny-8bit", nchans=64, f_top=1500.0, df=-1.0, dt=64e-6, nbits=8,
            nsamps=4096, ndm=32, dm_max=155.0, out="u32", dist="gauss", sigma=16,
            npulses=1, pulse_dm_index=10),
    2: _cfg(2, name="cfg2-survey-2bit", nchans=1024, f_top=1581.8, df=-0.390625, dt=64e-6, nbits=2,
            nsamps=1 << 19, ndm=1200, dm_max=1000.0, out="f32", dist="uniform"),
    3: _cfg(3, name="cfg3-lowfreq-8bit", nchans=4096, f_top=400.0, df=-0.0244140625, dt=64e-6, nbits=8,
            nsamps=1 << 20, ndm=1024, dm_max=500.0, out="f32", dist="gauss", sigma=20, npulses=8),
    4: _cfg(4, name="cfg4-widedm-4bit", nchans=1024, f_top=1581.8, df=-0.390625, dt=64e-6, nbits=4,
            nsamps=1 << 20, ndm=4096, dm_max=2000.0, out="u16", dist="uniform"),
    5: _cfg(5, name="cfg5-13beam-8bit", nchans=1024, f_top=1581.8, df=-0.390625, dt=64e-6, nbits=8,
            nsamps=1 << 18, ndm=1200, dm_max=1000.0, out="f32", dist="gauss", sigma=16, nbeams=13),
}


# --------------------------------------------------------------------------- hash

def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right of int64 bit patterns."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def hash64(seed: int, beam, c: torch.Tensor, t: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser of a linear combination of (seed+1000*beam, c, t); int64 bit patterns.

    `beam` may be an int or an int64 tensor broadcastable with c and t.
    """
    if isinstance(beam, int):
        sb = _s64((seed + 1000 * beam) * _G0)
    else:
        sb = (seed + 1000 * beam) * _s64(_G0)
    x = sb + c * _s64(_G1) + t * _s64(_G2)
    x = (x ^ _lsr(x, 30)) * _s64(_G1)
    x = (x ^ _lsr(x, 27)) * _s64(_G2)
    return x ^ _lsr(x, 31)


def hash64_py(seed: int, beam: int, c: int, t: int) -> int:
    """The same function on Python integers (reference for the torch version; used by tests)."""
    x = ((seed + 1000 * beam) * _G0 + c * _G1 + t * _G2) & _MASK64
    x = ((x ^ (x >> 30)) * _G1) & _MASK64
    x = ((x ^ (x >> 27)) * _G2) & _MASK64
    return x ^ (x >> 31)


def _base_values(cfg: Config, beam, c: torch.Tensor, t: torch.Tensor) -> torch.Tensor:
    """Pulse-free sample values (int64 tensor, broadcast shape of c and t)."""
    h = hash64(cfg.seed, beam, c, t)
    if cfg.dist == "uniform":
        return _lsr(h, 64 - cfg.nbits)
    if cfg.dist == "gauss":
        s = h & 0xFF
        for k in range(1, 8):
            s = s + (_lsr(h, 8 * k) & 0xFF)
        num = (s - _IH_MEAN) * (cfg.sigma * 10000)
        den = _IH_SIGMA_X1E4
        v = 128 + torch.div(2 * num + den, 2 * den, rounding_mode="floor")
        return torch.clamp(v, 0, 255)
    raise ValueError(cfg.dist)


# ------------------------------------------------------------------------- pulses

@dataclass(frozen=True)
class Pulses:
    """Injected dispersed pulses: for pulse i, every channel c gets +amp at t0[i] + tracks[i][c].

    `tracks` are delay-table rows supplied by the caller (oracle rows in the tests);
    `dm_index[i]` records which DM trial each row belongs to.
    """
    dm_index: np.ndarray      # [npulses] int64
    t0: np.ndarray            # [npulses] int64
    tracks: np.ndarray        # [npulses][nchans] int64
    amp: int


def pulse_positions(cfg: Config, beam: int = 0) -> tuple[np.ndarray, np.ndarray]:
    """Seed-chosen (dm_index, t0) of the injected pulses (no delays involved)."""
    if cfg.npulses == 0:
        return np.zeros(0, np.int64), np.zeros(0, np.int64)
    dm_idx, t0 = [], []
    for i in range(cfg.npulses):
        h = hash64_py(cfg.seed ^ 0x5EED, beam, 1 << 20, i)
        if cfg.pulse_dm_index is not None and cfg.npulses == 1:
            dm_idx.append(cfg.pulse_dm_index)
        else:
            dm_idx.append((h >> 32) % cfg.ndm)
        t0.append((h & 0xFFFFFFFF) % cfg.nsamps)
    return np.asarray(dm_idx, np.int64), np.asarray(t0, np.int64)


def make_pulses(cfg: Config, delay_rows_for, beam: int = 0) -> Optional[Pulses]:
    """Build the Pulses of `cfg`; `delay_rows_for(dm_indices) -> int64 [n][nchans]` is the caller's table."""
    if cfg.npulses == 0:
        return None
    dm_idx, t0 = pulse_positions(cfg, beam)
    tracks = np.asarray(delay_rows_for(dm_idx), dtype=np.int64).reshape(cfg.npulses, cfg.nchans)
    return Pulses(dm_index=dm_idx, t0=t0, tracks=tracks, amp=cfg.pulse_amp)


# --------------------------------------------------------------------- generation

def values_at(cfg: Config, beam, c, t, pulses: Optional[Pulses] = None,
              device: str | torch.device = "cpu") -> torch.Tensor:
    """Sample values at arbitrary (beam, c, t) points (broadcast), as an int64 tensor on `device`."""
    c = torch.as_tensor(c, dtype=torch.int64, device=device)
    t = torch.as_tensor(t, dtype=torch.int64, device=device)
    if not isinstance(beam, int):
        beam = torch.as_tensor(beam, dtype=torch.int64, device=device)
    v = _base_values(cfg, beam, c, t)
    if pulses is not None:
        vmax = (1 << cfg.nbits) - 1
        tracks = torch.as_tensor(pulses.tracks, dtype=torch.int64, device=device)
        for i in range(len(pulses.t0)):
            hit = (t == int(pulses.t0[i]) + tracks[i][c])
            v = torch.where(hit, torch.clamp(v + pulses.amp, max=vmax), v)
    return v


def gen_block(cfg: Config, beam: int, c_lo: int, c_hi: int, t_lo: int, t_hi: int,
              pulses: Optional[Pulses] = None, device: str | torch.device = "cpu") -> torch.Tensor:
    """Unpacked samples in[beam][c_lo:c_hi][t_lo:t_hi] as a uint8 tensor on `device`."""
    c = torch.arange(c_lo, c_hi, dtype=torch.int64, device=device)[:, None]
    t = torch.arange(t_lo, t_hi, dtype=torch.int64, device=device)[None, :]
    return values_at(cfg, beam, c, t, pulses, device).to(torch.uint8)


def pack_rows(samples: torch.Tensor, nbits: int) -> torch.Tensor:
    """Pack uint8 samples [..., n] (n * nbits % 8 == 0) along the last axis, LSB first (R9)."""
    if nbits == 8:
        return samples.contiguous()
    per = 8 // nbits
    n = samples.shape[-1]
    assert n % per == 0, "row length must fill whole bytes"
    s = samples.reshape(*samples.shape[:-1], n // per, per).to(torch.int32)
    out = torch.zeros(s.shape[:-1], dtype=torch.int32, device=samples.device)
    for k in range(per):
        out |= s[..., k] << (k * nbits)
    return out.to(torch.uint8)


def row_layout(cfg: Config, max_delay: int) -> tuple[int, int]:
    """(samples per row rounded to a 16-byte multiple, row stride in bytes) for nsamps + max_delay samples."""
    nsamp_in = cfg.nsamps + int(max_delay)
    row_bytes = (nsamp_in * cfg.nbits + 7) // 8
    stride = (row_bytes + 15) // 16 * 16
    return stride * 8 // cfg.nbits, stride


def gen_packed(cfg: Config, max_delay: int, pulses: Optional[Pulses] = None,
               device: str | torch.device = "cpu", beams: Optional[Sequence[int]] = None,
               chan_chunk: int = 64) -> tuple[torch.Tensor, int]:
    """The packed input in[beam][c][byte] (uint8, shape [nbeams][nchans][stride]) and its row stride in bytes.

    Rows hold nsamps + max_delay samples and are filled with generated samples out
    to the 16-byte padded stride (the padding is never addressed by a valid output).
    `max_delay` comes from the caller's delay table.
    """
    nsamp_row, stride = row_layout(cfg, max_delay)
    beams = list(range(cfg.nbeams)) if beams is None else list(beams)
    out = torch.empty((len(beams), cfg.nchans, stride), dtype=torch.uint8, device=device)
    for bi, b in enumerate(beams):
        for c0 in range(0, cfg.nchans, chan_chunk):
            c1 = min(cfg.nchans, c0 + chan_chunk)
            blk = gen_block(cfg, b, c0, c1, 0, nsamp_row, pulses, device)
            out[bi, c0:c1] = pack_rows(blk, cfg.nbits)
    return out, stride
