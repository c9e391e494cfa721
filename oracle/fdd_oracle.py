"""CPU oracle for Fourier-domain dedispersion (FDD) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl
reference`` legs may import this module.  It shares no code with the CUDA path
(``paper_2110_03482_b200/``) and imports nothing from it.

What it computes (Bassa et al., arXiv:2110.03482; line numbers are /root/reference/PAPER.md):

  O1  x[c][n]  = (double) in_u8[n][c], zero padded to N = next power of two >= N_t
                 (PAPER.md:149 input matrix; "zero padded ... power of two")
  O2  X[c][k]  = sum_n x[c][n] exp(-2 pi i k n / N), k = 0..N/2          (Eq. 3)
  O3  d[j][c]  = K dm_j (nu_c^-2 - nu_hi^-2) / tsamp   [samples]          (Eq. 1)
                 nu_c = linspace(f_lo, f_hi, N_nu)[c]; reference = highest channel
  O4  Y[j][k]  = sum_c X[c][k] exp(+2 pi i frac(k d[j][c] / N))            (Eq. 4 + Eq. 7)
  O5  y[j][n]  = (1/N) [ Re Y[j][0] + 2 sum_{k=1}^{N/2-1} Re(Y[j][k] e^{2 pi i k n/N})
                         + Re(Y[j][N/2]) (-1)^n ],  n < N_t                (Eq. 6)
  O6  TIME output = y;  FOURIER output = Y (unnormalised);
      valid = N_t - ceil(max |d|)

Readings of the paper taken here:
  S1  sign: the semantics are y_dm[n] = sum_nu x_nu[(n + d) mod N] (an *advance* by the
      dispersion delay: "peaks being aligned", PAPER.md:96 wrap puts samples from
      the start at the end).  With Eq. 3's forward kernel e^{-2 pi i f t} that is the phasor
      e^{+2 pi i k d / N}.  Eq. 4's literal minus sign belongs to the opposite transform sign;
      for real input the two conventions give conjugate spectra and identical time series.
  S5  K = 4.148808e3 MHz^2 pc^-1 cm^3 s (BASELINE.json) unless overridden; the paper's
      (2.41e-4)^-1 differs by 1.4e-4 relative.
  S6  TIME output carries the 1/N of the inverse transform (DM = 0 is the plain channel sum).
  S7  delays are applied unrounded (band-limited fractional shift), unlike Eq. 2's rounding.
  S8  for even N an inverse *real* transform uses only Re Y[N/2] (and Re Y[0]).
  S10 valid length uses ceil(max|d| (1 - 1e-12)) so that mathematically integer delays that
      evaluate to 255.00000000000003 do not flip the ceil.

Two tiers, same steps:
  * naive tier      O2 / O5 as literal O(N^2) sums (dense DFT matrix with the exponent k*n
                    reduced mod N in integers)   -- ``fdd_naive``
  * at-scale tier   O2 / O5 replaced by numpy's fp64 FFT (pocketfft), validated against the
                    naive tier in tests/test_oracle_pins.py -- ``fdd_fft``, ``fdd_rows``;
                    and single bins straight from the definition -- ``single_bins``.
All arithmetic is IEEE double; the phase product k*d/N is formed in long double and reduced
to a fraction of a cycle before the cast (phases reach 2e4 cycles in config 5).

Pins (tests/test_oracle_pins.py): P1 DFT vs library rfft; P2 DM=0 is the channel sum; P3
integer delays == circular shift-and-sum in integer arithmetic; P4 fractional delays ==
brute-force periodic-sinc interpolation in the time domain; P5 injected pulse peaks at its
trial; P6 Parseval / |Y|=|X|; P7 DC invariance; P8 Eq. 5 <-> Eq. 6 and shift covariance;
P9 pure tone at 1.9e4 cycles; P10 tiers agree.  No function here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import math
import os
from typing import Iterable, Optional, Sequence

import numpy as np

K_DM_DEFAULT = 4.148808e3   # S5


# ----------------------------------------------------------------------------- O3 / O6
def next_pow2(n: int) -> int:
    """N of PAPER.md:155 ("zero padded such that the number of samples becomes a power of two")."""
    n = int(n)
    if n < 1:
        raise ValueError("nsamps must be >= 1")
    return 1 << (n - 1).bit_length()


def channel_freqs(nchans: int, f_lo: float, f_hi: float) -> np.ndarray:
    """nu_c: channel centres evenly spaced from f_lo to f_hi inclusive (reading S3)."""
    if nchans == 1:
        return np.array([f_hi], dtype=np.float64)
    c = np.arange(nchans, dtype=np.float64)
    return f_lo + c * (f_hi - f_lo) / (nchans - 1)


def delay_table(nchans: int, f_lo: float, f_hi: float, tsamp: float, dm_list: Sequence[float],
                k_dm: float = K_DM_DEFAULT) -> np.ndarray:
    """d[j][c] in samples, Eq. 1 against the highest channel."""
    nu = channel_freqs(nchans, f_lo, f_hi)
    per_dm = k_dm * (nu ** -2 - float(f_hi) ** -2) / tsamp          # samples per unit DM
    dm = np.asarray(dm_list, dtype=np.float64)
    return dm[:, None] * per_dm[None, :]


def valid_length(delays: np.ndarray, nsamps: int) -> int:
    """O6 / S10: samples not contaminated by the cyclic wrap."""
    dmax = float(np.max(np.abs(delays))) if delays.size else 0.0
    return int(nsamps - math.ceil(dmax * (1.0 - 1e-12)))


# ----------------------------------------------------------------------------- O1
def unpack(in_u8: np.ndarray, nfft: Optional[int] = None) -> np.ndarray:
    """O1: x[c][n] as float64, zero padded to nfft."""
    in_u8 = np.asarray(in_u8)
    nsamps, nchans = in_u8.shape
    n = next_pow2(nsamps) if nfft is None else int(nfft)
    x = np.zeros((nchans, n), dtype=np.float64)
    x[:, :nsamps] = in_u8.T
    return x


# ----------------------------------------------------------------------------- O2 (naive)
def naive_rdft(x: np.ndarray, block: int = 256) -> np.ndarray:
    """O2: X[c][k] = sum_n x[c][n] exp(-2 pi i k n / N), k = 0..N/2, by the definition (Eq. 3).

    The exponent k*n is reduced mod N in integer arithmetic so the twiddle is exact to fp64.
    """
    x = np.asarray(x, dtype=np.float64)
    n = x.shape[-1]
    nb = n // 2 + 1
    idx = np.arange(n, dtype=np.int64)
    out = np.empty(x.shape[:-1] + (nb,), dtype=np.complex128)
    for k0 in range(0, nb, block):
        k = np.arange(k0, min(k0 + block, nb), dtype=np.int64)
        ang = (-2.0 * np.pi / n) * ((k[:, None] * idx[None, :]) % n)   # [kb][n]
        w = np.cos(ang) + 1j * np.sin(ang)
        out[..., k0:k0 + k.size] = x @ w.T
    return out


# ----------------------------------------------------------------------------- O4
def phasor(k: np.ndarray, d: float, nfft: int) -> np.ndarray:
    """exp(+2 pi i k d / N) with k*d/N reduced to a fraction of a cycle in long double (Eq. 4, S1)."""
    cyc = np.asarray(k, dtype=np.longdouble) * np.longdouble(d) / np.longdouble(nfft)
    frac = (cyc - np.rint(cyc)).astype(np.float64)
    ang = 2.0 * np.pi * frac
    return np.cos(ang) + 1j * np.sin(ang)


def phase_rotate_sum(X: np.ndarray, delays: np.ndarray, nfft: int,
                     bins: Optional[np.ndarray] = None) -> np.ndarray:
    """O4: Y[j][k] = sum_c X[c][k] exp(+2 pi i k d[j][c] / N)  (Eq. 7).

    ``X`` is [nchans][len(bins)]; ``bins`` gives the bin number k of each column (default 0..N/2).
    """
    X = np.asarray(X, dtype=np.complex128)
    nchans, nb = X.shape
    k = np.arange(nb, dtype=np.int64) if bins is None else np.asarray(bins, dtype=np.int64)
    delays = np.asarray(delays, dtype=np.float64)
    ndm = delays.shape[0]
    Y = np.zeros((ndm, nb), dtype=np.complex128)
    for j in range(ndm):
        acc = np.zeros(nb, dtype=np.complex128)
        for c in range(nchans):
            acc += X[c] * phasor(k, delays[j, c], nfft)
        Y[j] = acc
    return Y


_C_LIB = None


def _c_lib():
    """oracle/_fdd_oracle_c.so (built by ``python -m oracle.build``), or None if not built."""
    global _C_LIB
    if _C_LIB is None:
        path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "_fdd_oracle_c.so")
        if not os.path.exists(path):
            return None
        lib = ctypes.CDLL(path)
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_phase_rotate_sum.restype = None
        lib.oracle_phase_rotate_sum.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                                ctypes.c_int64, ctypes.c_int64, ctypes.c_int64,
                                                ctypes.c_int64, ctypes.c_int, ctypes.c_void_p]
        _C_LIB = lib
    return _C_LIB


def num_threads() -> int:
    """Threads the C part of the oracle uses (1 when it is not built)."""
    lib = _c_lib()
    return int(lib.oracle_num_threads()) if lib is not None else 1


def phase_rotate_sum_c(X: np.ndarray, delays: np.ndarray, nfft: int,
                       bins: Optional[np.ndarray] = None, out: Optional[np.ndarray] = None,
                       accumulate: bool = False) -> np.ndarray:
    """O4 again, as the plain C loops of fdd_oracle_c.c (same definition, long-double phase).

    Used by the at-scale tier where the numpy version would take minutes; pinned to the numpy
    version in tests.  Falls back to the numpy version when the C library is not built.
    """
    X = np.ascontiguousarray(X, dtype=np.complex128)
    delays = np.ascontiguousarray(delays, dtype=np.float64)
    nchans, nb = X.shape
    nrows = delays.shape[0]
    assert delays.shape == (nrows, nchans)
    lib = _c_lib()
    if lib is None:
        Y = phase_rotate_sum(X, delays, nfft, bins)
        if out is not None:
            out[...] = out + Y if accumulate else Y
            return out
        return Y
    if out is None:
        out = np.zeros((nrows, nb), dtype=np.complex128)
        accumulate = False
    assert out.shape == (nrows, nb) and out.dtype == np.complex128 and out.flags.c_contiguous
    b = None
    if bins is not None:
        b = np.ascontiguousarray(bins, dtype=np.int64)
        assert b.shape == (nb,)
    lib.oracle_phase_rotate_sum(X.ctypes.data, delays.ctypes.data,
                                b.ctypes.data if b is not None else None,
                                nchans, nb, nrows, int(nfft), int(bool(accumulate)),
                                out.ctypes.data)
    return out


# ----------------------------------------------------------------------------- O5 (naive)
def naive_irdft(Y: np.ndarray, nfft: int, nsamps: int, block: int = 256) -> np.ndarray:
    """O5: inverse real DFT by the definition, using only Re of bins 0 and N/2 (Eq. 6, S6, S8)."""
    Y = np.asarray(Y, dtype=np.complex128)
    n = int(nfft)
    assert n % 2 == 0 and Y.shape[-1] == n // 2 + 1
    k = np.arange(1, n // 2, dtype=np.int64)
    out = np.empty(Y.shape[:-1] + (nsamps,), dtype=np.float64)
    for n0 in range(0, nsamps, block):
        t = np.arange(n0, min(n0 + block, nsamps), dtype=np.int64)
        ang = (2.0 * np.pi / n) * ((k[:, None] * t[None, :]) % n)       # [k][t]
        cr, sn = np.cos(ang), np.sin(ang)
        mid = 2.0 * (Y[..., 1:n // 2].real @ cr - Y[..., 1:n // 2].imag @ sn)
        sign = np.where(t % 2 == 0, 1.0, -1.0)
        out[..., n0:n0 + t.size] = (Y[..., :1].real + mid + Y[..., n // 2:].real * sign) / n
    return out


# ----------------------------------------------------------------------------- O5' (next row f3)
def naive_irdft_reduced(Y: np.ndarray, nfft: int, nsamps: int, log2_factor: int,
                        block: int = 256) -> np.ndarray:
    """Down-sampling "by reducing the length of the inverse Fourier transform".

    The spectrum is cut at the new Nyquist bin, M = nfft / 2^m points instead of nfft:
        y_m[n] = (1/nfft) [Re Y_0 + 2 sum_{k=1}^{M/2-1} Re(Y_k e^{2 pi i k n / M}) + Re(Y_{M/2}) (-1)^n]
    for n < ceil(nsamps / 2^m): the ideal low-pass of the full-rate series y sampled every 2^m
    samples, in the units of y (scaling 1/nfft as in O5; only Re of the two edge bins, S8).
    """
    Y = np.asarray(Y, dtype=np.complex128)
    n, m = int(nfft), int(log2_factor)
    M = n >> m
    assert m >= 0 and M >= 2 and Y.shape[-1] >= M // 2 + 1
    nout = -(-int(nsamps) // (1 << m))
    k = np.arange(1, M // 2, dtype=np.int64)
    out = np.empty(Y.shape[:-1] + (nout,), dtype=np.float64)
    for n0 in range(0, nout, block):
        t = np.arange(n0, min(n0 + block, nout), dtype=np.int64)
        ang = (2.0 * np.pi / M) * ((k[:, None] * t[None, :]) % M)
        cr, sn = np.cos(ang), np.sin(ang)
        mid = 2.0 * (Y[..., 1:M // 2].real @ cr - Y[..., 1:M // 2].imag @ sn)
        sign = np.where(t % 2 == 0, 1.0, -1.0)
        out[..., n0:n0 + t.size] = (Y[..., :1].real + mid + Y[..., M // 2:M // 2 + 1].real * sign) / n
    return out


def irfft_reduced(Y: np.ndarray, nfft: int, nsamps: int, log2_factor: int) -> np.ndarray:
    """At-scale tier of naive_irdft_reduced (numpy fp64 FFT; validated against it in the pins)."""
    n, m = int(nfft), int(log2_factor)
    M = n >> m
    nout = -(-int(nsamps) // (1 << m))
    Yt = np.array(np.asarray(Y, dtype=np.complex128)[..., :M // 2 + 1])
    # numpy's irfft normalises by 1/M; the definition above by 1/nfft
    return np.fft.irfft(Yt, n=M, axis=-1)[..., :nout] * (M / n)


# ----------------------------------------------------------------------------- whole path
def fdd_naive(in_u8: np.ndarray, delays: np.ndarray, mode: str = "time") -> np.ndarray:
    """O1..O6 with literal O(N^2) transforms.  Small inputs only (N <= 8192)."""
    nsamps = in_u8.shape[0]
    n = next_pow2(nsamps)
    X = naive_rdft(unpack(in_u8, n))
    Y = phase_rotate_sum(X, delays, n)
    if mode == "fourier":
        return Y
    return naive_irdft(Y, n, nsamps)


def fdd_fft(in_u8: np.ndarray, delays: np.ndarray, mode: str = "time") -> np.ndarray:
    """At-scale tier: O2/O5 by numpy's fp64 FFT (validated against fdd_naive, pin P10)."""
    nsamps = in_u8.shape[0]
    n = next_pow2(nsamps)
    X = np.fft.rfft(unpack(in_u8, n), axis=-1)
    Y = phase_rotate_sum(X, delays, n)
    if mode == "fourier":
        return Y
    return np.fft.irfft(Y, n=n, axis=-1)[..., :nsamps]


def fdd_rows(in_u8: np.ndarray, delays: np.ndarray, rows: Iterable[int], mode: str = "time",
             chan_block: int = 32, log2_factor: int = 0) -> np.ndarray:
    """At-scale tier for a subset of DM rows, channel block by channel block (memory-light).

    Same O1..O6 as fdd_fft; only the loop order differs (channels outermost) so that a
    1024 x 2^20 input never has to exist as complex128 all at once.
    """
    rows = list(rows)
    nsamps, nchans = in_u8.shape
    n = next_pow2(nsamps)
    nb = n // 2 + 1
    d = np.asarray(delays, dtype=np.float64)[rows]
    Y = np.zeros((len(rows), nb), dtype=np.complex128)
    for c0 in range(0, nchans, chan_block):
        c1 = min(c0 + chan_block, nchans)
        X = np.fft.rfft(unpack(in_u8[:, c0:c1], n), axis=-1)
        phase_rotate_sum_c(X, d[:, c0:c1], n, out=Y, accumulate=True)
    return rows_from_spectrum(Y, n, nsamps, mode, log2_factor)


def rows_from_spectrum(Y: np.ndarray, nfft: int, nsamps: int, mode: str = "time",
                       log2_factor: int = 0) -> np.ndarray:
    """O5 + O6 of the at-scale tier: the output rows that belong to the sums Y[j][0..N/2] of O4.

    The last step of ``fdd_rows``, callable on its own so that tests which need the TIME, FOURIER
    and reduced-length (row f3) outputs of the same DM rows run O1..O4 once.
    """
    n = int(nfft)
    if log2_factor:
        if mode == "fourier":
            return Y[..., :(n >> log2_factor) // 2 + 1]
        return irfft_reduced(Y, n, nsamps, log2_factor)
    if mode == "fourier":
        return Y
    return np.fft.irfft(Y, n=n, axis=-1)[..., :nsamps]


def single_bins(in_u8: np.ndarray, delays: np.ndarray, bins: Sequence[int],
                rows: Optional[Iterable[int]] = None, time_block: int = 1 << 14) -> np.ndarray:
    """Y[j][k] for a handful of bins k straight from the definitions O1+O2+O4 (no FFT).

    PAPER.md:84: "the data for each spin frequency need to be processed independently" --
    so single bins of the FOURIER output can be checked at full size at O(N_nu N_t) each.
    """
    nsamps, nchans = in_u8.shape
    n = next_pow2(nsamps)
    bins = np.asarray(list(bins), dtype=np.int64)
    X = np.zeros((nchans, bins.size), dtype=np.complex128)
    for n0 in range(0, nsamps, time_block):
        t = np.arange(n0, min(n0 + time_block, nsamps), dtype=np.int64)
        ang = (-2.0 * np.pi / n) * ((bins[:, None] * t[None, :]) % n)    # [bins][t]
        w = np.cos(ang) + 1j * np.sin(ang)
        X += in_u8[n0:n0 + t.size].astype(np.float64).T @ w.T
    d = np.asarray(delays, dtype=np.float64)
    if rows is not None:
        d = d[list(rows)]
    return phase_rotate_sum_c(X, d, n, bins=bins)


# ----------------------------------------------------------------------------- next row f1
def fdd_beams(in_u8_beams: np.ndarray, delays: np.ndarray, rows: Optional[Iterable[int]] = None,
              mode: str = "time") -> np.ndarray:
    """Several beams with one delay table ("reusing phase rotations ... multiple
    beams"): the beams share nothing but the phasors, so the definition is O1..O6 beam by beam.

    ``in_u8_beams`` is [nbeams][nsamps][nchans]; returns [nbeams][rows][...] (at-scale tier).
    """
    in_u8_beams = np.asarray(in_u8_beams)
    assert in_u8_beams.ndim == 3
    rows = list(range(np.asarray(delays).shape[0])) if rows is None else list(rows)
    return np.stack([fdd_rows(b, delays, rows, mode=mode) for b in in_u8_beams])
