"""Seeded synthetic filterbanks shaped like the paper's data, and the five BASELINE.json configs.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's tests/bench.
It holds workload descriptions and input generation only -- none of the method's arithmetic
(no delay table, no decimation, no dedispersion) and it imports neither `oracle` nor the
C-ABI binding.  The dispersed-pulse injector evaluates the cold-plasma sweep (PAPER.md:258,
Eq. 1.1) in its own float expression purely to *shape the input signal*, the way the thesis
injects simulated pulses into 8-bit data; neither side reads those values.

Shapes follow PAPER.md:303, :351, :389 (4096 channels, one spectrum per 1.31072 ms, 8-bit
samples) and BASELINE.json `configs`.  The inputs stand in for SPOTLIGHT beam data, which is
not available here.  Recipe:
  noise  = clip(rint(normal(mean, sd)), 0, 2^bits - 1), generated per 16-channel block from
           numpy Generator(PCG64(SeedSequence([seed, beam, block]))) in float32;
  pulses = +height on `width` consecutive samples starting at t0 + round(sweep(c)), then clip;
  zeroed = a seeded 2 % subset of channel rows set to 0 (RFI-flagged channels, config 3).
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

_BLOCK = 16  # channels per independently seeded block


@dataclass(frozen=True)
class DMRange:
    dm_lo: float
    dm_step: float
    ndm: int
    decim: int


@dataclass(frozen=True)
class Pulse:
    dm: float
    t0: int
    width: int
    height: int


@dataclass(frozen=True)
class Workload:
    name: str
    f_top_mhz: float
    chan_width_mhz: float
    nchans: int
    tsamp_s: float
    nsamps: int
    nbeams: int
    in_bits: int
    ranges: Tuple[DMRange, ...]
    seed: int
    noise_mean: float
    noise_sd: float
    zero_frac: float = 0.0
    n_pulses: int = 0          # random pulses per beam (drawn from the seed)
    pulse_dm: Tuple[float, float] = (0.0, 0.0)
    pulse_height: int = 30
    fixed_pulses: Tuple[Pulse, ...] = field(default_factory=tuple)
    max_sweep: int = 0         # largest delay of the plan in input samples (bounds pulse t0)

    @property
    def dtype(self):
        return np.uint8 if self.in_bits == 8 else np.uint16

    @property
    def total_trials(self) -> int:
        return sum(r.ndm for r in self.ranges)

    @property
    def in_bytes(self) -> int:
        return self.nbeams * self.nchans * self.nsamps * (self.in_bits // 8)


def make_ranges(spec: List[Tuple[float, float, float, int]]) -> Tuple[DMRange, ...]:
    """Harness rule for trial counts (reading A7): non-final ranges are half-open,
    ndm = round((hi-lo)/step); the final range includes its upper end (+1)."""
    out = []
    for i, (lo, hi, step, decim) in enumerate(spec):
        n = int(round((hi - lo) / step)) + (1 if i == len(spec) - 1 else 0)
        out.append(DMRange(float(lo), float(step), n, int(decim)))
    return tuple(out)


def _w(name, f_top, bw, nchans, tsamp, nsamps, nbeams, bits, ranges, seed, mean, sd, **kw):
    return Workload(name, float(f_top), -float(bw) / nchans, nchans, float(tsamp), int(nsamps), nbeams, bits,
                    make_ranges(ranges), seed, float(mean), float(sd), **kw)


# BASELINE.json configs[0..4] (1-based names as in SURVEY.md section 8).
CONFIGS = {
    1: _w("cfg1_tiny_128ch", 500.0, 200.0, 128, 1.024e-3, 8192, 1, 8, [(0, 100, 1.0, 1)], 353101, 128, 10,
          fixed_pulses=(Pulse(50.0, 1024, 4, 40),), max_sweep=2835),
    2: _w("cfg2_1024ch", 750.0, 200.0, 1024, 655.36e-6, 2 ** 17, 1, 8, [(0, 500, 0.5, 1)], 353102, 128, 16,
          n_pulses=5, pulse_dm=(20.0, 480.0), max_sweep=4829),
    3: _w("cfg3_spotlight_4096ch", 750.0, 200.0, 4096, 1.31072e-3, 2 ** 18, 1, 8,
          [(0, 200, 0.1, 1), (200, 600, 0.2, 2), (600, 2000, 0.5, 4)], 353103, 128, 12, zero_frac=0.02),
    4: _w("cfg4_uint16_4096ch", 500.0, 200.0, 4096, 1.31072e-3, 2 ** 18, 1, 16,
          [(0, 1000, 0.25, 1), (1000, 3000, 1.0, 8)], 353104, 2 ** 15, 2 ** 10),
    5: _w("cfg5_32beams_2048ch", 750.0, 200.0, 2048, 1.31072e-3, 2 ** 16, 32, 8, [(0, 1000, 0.5, 1)], 353105, 128, 12,
          n_pulses=1, pulse_dm=(20.0, 980.0), max_sweep=4833),
}


def scaled(w: Workload, *, nchans=None, nsamps=None, nbeams=None, ranges=None, name=None) -> Workload:
    """A smaller/larger variant of a workload with the same band, statistics and seed."""
    nch = nchans or w.nchans
    bw = -w.chan_width_mhz * w.nchans
    return Workload(name or (w.name + "_scaled"), w.f_top_mhz, -bw / nch, nch, w.tsamp_s, nsamps or w.nsamps,
                    nbeams or w.nbeams, w.in_bits, tuple(ranges) if ranges is not None else w.ranges, w.seed,
                    w.noise_mean, w.noise_sd, w.zero_frac, w.n_pulses, w.pulse_dm, w.pulse_height,
                    w.fixed_pulses, w.max_sweep)


def pulses_for_beam(w: Workload, beam: int) -> Tuple[Pulse, ...]:
    """The pulses injected into one beam: the fixed ones plus n_pulses drawn from the seed."""
    out = list(w.fixed_pulses)
    if w.n_pulses:
        rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([w.seed, beam, 1 << 20])))
        hi_t0 = max(1, w.nsamps - w.max_sweep - 16)
        for _ in range(w.n_pulses):
            dm = float(rng.uniform(*w.pulse_dm))
            width = int(rng.integers(1, 17))
            t0 = int(rng.integers(0, hi_t0))
            out.append(Pulse(dm, t0, width, w.pulse_height))
    return tuple(out)


def zeroed_channels(w: Workload, beam: int) -> np.ndarray:
    """Sorted indices of the channel rows set to zero (RFI-flagged), chosen without replacement."""
    n = int(round(w.zero_frac * w.nchans))
    if n == 0:
        return np.empty(0, dtype=np.int64)
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([w.seed, beam, (1 << 20) + 1])))
    return np.sort(rng.choice(w.nchans, size=n, replace=False))


def _sweep_samples(w: Workload, dm: float) -> np.ndarray:
    """Arrival-time sweep of a dispersed pulse in input samples, per channel (signal synthesis only)."""
    f = w.f_top_mhz + w.chan_width_mhz * np.arange(w.nchans, dtype=np.float64)
    return np.rint(4.148808e3 * dm * (f ** -2.0 - w.f_top_mhz ** -2.0) / w.tsamp_s).astype(np.int64)


def _noise_block(w: Workload, beam: int, block: int, out: np.ndarray) -> None:
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([w.seed, beam, block])))
    rows = out[block * _BLOCK:(block + 1) * _BLOCK]
    g = rng.standard_normal(rows.shape, dtype=np.float32)
    g *= np.float32(w.noise_sd)
    g += np.float32(w.noise_mean)
    np.rint(g, out=g)
    np.clip(g, 0, float(2 ** w.in_bits - 1), out=g)
    rows[...] = g.astype(w.dtype)


def generate_beam(w: Workload, beam: int = 0, out: np.ndarray | None = None, threads: int = 8) -> np.ndarray:
    """One beam's filterbank, [nchans][nsamps], uint8 or uint16, time contiguous."""
    if out is None:
        out = np.empty((w.nchans, w.nsamps), dtype=w.dtype)
    nblocks = (w.nchans + _BLOCK - 1) // _BLOCK
    if threads > 1 and nblocks > 1:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(lambda b: _noise_block(w, beam, b, out), range(nblocks)))
    else:
        for b in range(nblocks):
            _noise_block(w, beam, b, out)
    top = 2 ** w.in_bits - 1
    for p in pulses_for_beam(w, beam):
        sweep = _sweep_samples(w, p.dm)
        for c in range(w.nchans):
            a = p.t0 + int(sweep[c])
            b = min(a + p.width, w.nsamps)
            if a < w.nsamps:
                seg = out[c, a:b].astype(np.int64) + p.height
                out[c, a:b] = np.clip(seg, 0, top).astype(w.dtype)
    for c in zeroed_channels(w, beam):
        out[c, :] = 0
    return out


def generate(w: Workload, threads: int = 8) -> np.ndarray:
    """All beams, [nbeams][nchans][nsamps]."""
    x = np.empty((w.nbeams, w.nchans, w.nsamps), dtype=w.dtype)
    for b in range(w.nbeams):
        generate_beam(w, b, out=x[b], threads=threads)
    return x
