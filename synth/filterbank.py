"""Seeded synthetic 8-bit filterbank inputs (shared by the oracle tests, the GPU tests and bench.py).

This module holds *no* dedispersion arithmetic: it only simulates what a telescope
records -- white noise per (time, channel) sample plus dispersed pulses that arrive
later at lower observing frequency (cold-plasma law, Eq. 1) -- and
names the five workload configurations of BASELINE.json.  It imports neither
``oracle`` nor the CUDA package, and neither of those shares code with it beyond
calling these generators.

The inputs stand in for the paper's simulated datasets (5 min of
64 us samples, 1024 channels, N_DM = 128...4096), which were never published.

Layout: ``uint8 [nsamps][nchans]``, channel fastest, channel 0 = lowest frequency
(time-major filterbank order).

Recipe:
  noise  z ~ N(0,1) from numpy ``default_rng(seed)`` (PCG64), float32, drawn in
         row blocks of ``ROWS_PER_BLOCK`` time samples, channel fastest;
  value  = clip(rint(128 + 16 z + pulses), 0, 255)     (round-half-even)
  pulse  = amp * exp(-(t - t_c)^2 / (2 sigma^2)), sigma = FWHM / 2.35482,
           t_c = t0 + K * DM * (nu^-2 - nu_hi^-2) / tsamp  (unrounded, in samples),
           added to the float noise before rounding; samples outside [0, nsamps)
           are dropped (no wrap).
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional, Sequence, Tuple

import numpy as np

K_DM = 4.148808e3          # MHz^2 pc^-1 cm^3 s  (BASELINE.json north_star)
ROWS_PER_BLOCK = 4096      # part of the recipe: noise is drawn block by block
_FWHM_TO_SIGMA = 1.0 / (2.0 * math.sqrt(2.0 * math.log(2.0)))


@dataclasses.dataclass(frozen=True)
class Pulse:
    t0: float          # arrival sample at the highest channel
    dm: float          # pc cm^-3
    fwhm: float        # samples
    amp: float         # input units, per channel


@dataclasses.dataclass(frozen=True)
class Workload:
    name: str
    seed: int
    nchans: int
    f_lo: float        # MHz, centre of channel 0
    f_hi: float        # MHz, centre of channel nchans-1
    tsamp: float       # s
    nsamps: int
    dm_list: Tuple[float, ...]
    mode: str          # "time" | "fourier"
    pulses: Tuple[Pulse, ...]

    @property
    def ndm(self) -> int:
        return len(self.dm_list)

    def freqs(self) -> np.ndarray:
        if self.nchans == 1:
            return np.array([self.f_hi], dtype=np.float64)
        return np.linspace(self.f_lo, self.f_hi, self.nchans, dtype=np.float64)


def one_sample_dm_step(f_lo: float, f_hi: float, tsamp: float) -> float:
    """DM step that smears by exactly one sample across the band (BASELINE.json configs 2-4)."""
    return tsamp / (K_DM * (f_lo ** -2 - f_hi ** -2))


def _seeded_pulses(seed: int, n: int, nsamps: int, dm_lo: float, dm_hi: float,
                   fwhm: float, amp: float) -> List[Pulse]:
    rng = np.random.default_rng(seed + 7919)
    t0 = rng.uniform(0.05 * nsamps, 0.6 * nsamps, size=n)
    dm = rng.uniform(dm_lo, dm_hi, size=n)
    return [Pulse(float(a), float(b), fwhm, amp) for a, b in zip(t0, dm)]


def _pulse_train(period_samples: float, nsamps: int, dm: float, fwhm: float, amp: float,
                 phase0: float) -> List[Pulse]:
    out = []
    t = phase0
    while t < nsamps:
        out.append(Pulse(t, dm, fwhm, amp))
        t += period_samples
    return out


def workload(name: str, ndm: Optional[int] = None) -> Workload:
    """The five BASELINE.json configs as concrete seeded inputs.

    ``ndm`` overrides the trial count for the config-4 DM sweep ("sweep").
    """
    if name in ("tiny", "config1"):
        dms = tuple(2.0 * i for i in range(32))
        return Workload("tiny", 1001, 64, 1400.0, 1500.0, 64e-6, 8192, dms, "time",
                        (Pulse(2048.0, 30.0, 4.0, 40.0),))
    if name in ("config2", "config3", "sweep", "config4"):
        f_lo, f_hi, tsamp = 1200.0, 1500.0, 64e-6
        step = one_sample_dm_step(f_lo, f_hi, tsamp)
        if name == "config2":
            seed, nsamps, n = 1002, 1 << 18, 256
        else:
            seed, nsamps, n = 1003, 1 << 20, 1024
        if name in ("sweep", "config4"):
            n = 4096 if ndm is None else int(ndm)
        elif ndm is not None:
            n = int(ndm)
        dms = tuple(step * i for i in range(n))
        pulses = _seeded_pulses(seed, 5, nsamps, 0.0, 500.0, 4.0, 40.0)
        if seed == 1003:
            # force one pulse onto the trial grid (trial 40 of the one-sample step)
            pulses = pulses + [Pulse(0.25 * nsamps, step * 40, 4.0, 40.0)]
        label = {"config2": "config2", "config3": "config3"}.get(name, "config4_sweep")
        return Workload(label, seed, 1024, f_lo, f_hi, tsamp, nsamps, dms, "time", tuple(pulses))
    if name == "config5":
        tsamp, nsamps = 491.52e-6, 1 << 19
        n = 8192 if ndm is None else int(ndm)
        dms = tuple(0.01 * i for i in range(n))
        period = 0.714 / tsamp
        pulses = _pulse_train(period, nsamps, 26.8, 8.0, 6.0, phase0=100.0)
        return Workload("config5", 1005, 400, 110.0, 190.0, tsamp, nsamps, dms, "fourier",
                        tuple(pulses))
    if name == "paper":
        # The shape of the paper's own runs: 5 min of 64 us samples (4 687 500,
        # zero padded to 2^23), 1024 channels over 400 MHz below 1581 MHz, trial DMs 0, 2, 4, ...
        # The data themselves (simulated signals) were never published: seeded noise + pulses.
        nsamps, f_lo, f_hi, tsamp = 4687500, 1181.0, 1581.0, 64e-6
        n = 1024 if ndm is None else int(ndm)
        dms = tuple(2.0 * i for i in range(n))
        pulses = _seeded_pulses(1006, 5, nsamps, 0.0, 2.0 * (n - 1), 4.0, 40.0)
        return Workload("paper_5min", 1006, 1024, f_lo, f_hi, tsamp, nsamps, dms, "time",
                        tuple(pulses))
    raise KeyError(name)


def small_workload(seed: int, nchans: int, nsamps: int, ndm: int, *, f_lo: float = 1200.0,
                   f_hi: float = 1500.0, tsamp: float = 64e-6, dm_step: Optional[float] = None,
                   dm0: float = 0.0, mode: str = "time", npulses: int = 2) -> Workload:
    """A free-form seeded workload of the same family, for parity cases between the configs."""
    if dm_step is None:
        dm_step = one_sample_dm_step(f_lo, f_hi, tsamp) if nchans > 1 and f_lo < f_hi else 1.0
    dms = tuple(dm0 + dm_step * i for i in range(ndm))
    pulses = _seeded_pulses(seed, npulses, nsamps, 0.0, max(dms) if ndm else 0.0, 4.0, 40.0)
    return Workload(f"small_{seed}", seed, nchans, f_lo, f_hi, tsamp, nsamps, dms, mode,
                    tuple(pulses))


def _pulse_entries(w: Workload) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Sparse (row, channel, value) contributions of all pulses, sorted by row."""
    if not w.pulses:
        z = np.zeros(0, dtype=np.int64)
        return z, z, np.zeros(0, dtype=np.float32)
    nu = w.freqs()
    disp = K_DM * (nu ** -2 - w.f_hi ** -2) / w.tsamp        # samples per unit DM, per channel
    rows, chans, vals = [], [], []
    ch = np.arange(w.nchans, dtype=np.int64)
    for p in w.pulses:
        sigma = p.fwhm * _FWHM_TO_SIGMA
        half = int(math.ceil(6.0 * sigma))
        centre = p.t0 + p.dm * disp                           # [nchans], fractional samples
        base = np.floor(centre).astype(np.int64)
        for off in range(-half, half + 2):
            r = base + off
            v = p.amp * np.exp(-0.5 * ((r - centre) / sigma) ** 2)
            ok = (r >= 0) & (r < w.nsamps)
            rows.append(r[ok]); chans.append(ch[ok]); vals.append(v[ok].astype(np.float32))
    rows = np.concatenate(rows); chans = np.concatenate(chans); vals = np.concatenate(vals)
    order = np.argsort(rows, kind="stable")
    return rows[order], chans[order], vals[order]


def make_filterbank(w: Workload, out: Optional[np.ndarray] = None) -> np.ndarray:
    """uint8 [nsamps][nchans] for workload ``w``; deterministic in ``w.seed``."""
    if out is None:
        out = np.empty((w.nsamps, w.nchans), dtype=np.uint8)
    assert out.shape == (w.nsamps, w.nchans) and out.dtype == np.uint8
    rng = np.random.default_rng(w.seed)
    prow, pch, pval = _pulse_entries(w)
    for r0 in range(0, w.nsamps, ROWS_PER_BLOCK):
        r1 = min(r0 + ROWS_PER_BLOCK, w.nsamps)
        blk = rng.standard_normal((r1 - r0, w.nchans), dtype=np.float32)
        blk *= np.float32(16.0)
        blk += np.float32(128.0)
        if prow.size:
            lo, hi = np.searchsorted(prow, (r0, r1))
            if hi > lo:
                np.add.at(blk, (prow[lo:hi] - r0, pch[lo:hi]), pval[lo:hi])
        np.rint(blk, out=blk)
        np.clip(blk, 0.0, 255.0, out=blk)
        out[r0:r1] = blk.astype(np.uint8)
    return out


def integer_delay_table(seed: int, ndm: int, nchans: int, max_delay: int) -> np.ndarray:
    """float64 [ndm][nchans] of exact integer sample delays (SURVEY.md pin P3), row 0 all zero.

    Rows grow roughly quadratically towards low channels like a dispersion sweep, but every
    entry is an integer so that the result has an exact integer-arithmetic definition.
    """
    rng = np.random.default_rng(seed)
    c = np.arange(nchans, dtype=np.float64)
    shape = ((nchans - 1 - c) / max(nchans - 1, 1)) ** 2
    tab = np.empty((ndm, nchans), dtype=np.float64)
    for j in range(ndm):
        scale = max_delay * j / max(ndm - 1, 1)
        jitter = rng.integers(0, 3, size=nchans)
        tab[j] = np.minimum(np.rint(scale * shape) + (jitter if j else 0), max_delay)
    tab[0] = 0.0
    return tab


def integer_progression_delay_table(ndm: int, nchans: int, max_step: int, dm0: int = 0) -> np.ndarray:
    """float64 [ndm][nchans] of exact integer delays d[j][c] = (dm0 + j) * a_c (pin P3).

    a_c = rint(max_step * (nu_c^-2 - nu_hi^-2) / (nu_lo^-2 - nu_hi^-2)) on a 1200-1500 MHz band: an
    integer number of samples per trial, max_step in channel 0 and zero in the top channel, so every
    channel's delays are an arithmetic progression over the trials -- a uniform "DM grid" whose
    delays all happen to be whole samples.  The result then has an exact integer definition
    (a circular shift-and-sum) AND the plan qualifies for the kernels that need progressions.
    """
    nu = np.linspace(1200.0, 1500.0, nchans) if nchans > 1 else np.array([1500.0])
    shape = (nu ** -2 - 1500.0 ** -2) / (1200.0 ** -2 - 1500.0 ** -2)
    a = np.rint(max_step * shape)
    j = dm0 + np.arange(ndm, dtype=np.float64)
    return j[:, None] * a[None, :]
