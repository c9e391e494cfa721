"""CPU oracle for the time-domain comparator -- TEST INFRASTRUCTURE ONLY.

Time-domain ("brute force", "incoherent") dedispersion, Eq. 2 of the paper:

    I(t, DM) = sum_nu I(t - Delta t(nu, DM), nu),   the shift rounded "to the nearest time sample".

Readings: S1 fixes the direction -- the sum re-aligns the pulse at the arrival time of
the highest channel, y[n] = sum_c x_c[n + s_c] with s_c >= 0 below the reference frequency;
"nearest" is floor(d + 1/2) (ties up); samples past the end wrap around over the nsamps input
samples, like the Fourier-domain result does for power-of-two lengths, so that for integer delays
the two methods agree everywhere -- the last ceil(max delay) samples are invalid in
both.

Plain integer arithmetic (int64): results are exact.  Shares no code with the CUDA path; only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import it.
"""
from __future__ import annotations

from typing import Iterable, Optional

import numpy as np


def shifts(delays: np.ndarray) -> np.ndarray:
    """Delays in samples -> integer shifts, nearest sample (Eq. 2's rounding), int64 [ndm][nchans]."""
    return np.floor(np.asarray(delays, dtype=np.float64) + 0.5).astype(np.int64)


def tdd_loops(in_u8: np.ndarray, delays: np.ndarray) -> np.ndarray:
    """Eq. 2 by three nested Python loops (tiny inputs only): the definition, nothing else."""
    nsamps, nchans = in_u8.shape
    s = shifts(delays)
    out = np.zeros((s.shape[0], nsamps), dtype=np.int64)
    for j in range(s.shape[0]):
        for n in range(nsamps):
            acc = 0
            for c in range(nchans):
                acc += int(in_u8[(n + int(s[j, c])) % nsamps, c])
            out[j, n] = acc
    return out


def tdd_rows(in_u8: np.ndarray, delays: np.ndarray, rows: Optional[Iterable[int]] = None) -> np.ndarray:
    """Eq. 2 for the DM rows ``rows`` (all if None), one circular shift per (row, channel)."""
    nsamps, nchans = in_u8.shape
    s = shifts(delays)
    rows = list(range(s.shape[0])) if rows is None else list(rows)
    out = np.zeros((len(rows), nsamps), dtype=np.int64)
    for c in range(nchans):
        col = in_u8[:, c].astype(np.int64)
        for i, j in enumerate(rows):
            out[i] += np.roll(col, -int(s[j, c]))
    return out
