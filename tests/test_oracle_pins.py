"""Pins for the CPU oracle: closed forms, invariants, brute force.

Nothing here touches the CUDA path.  Each test nails one part of oracle/fdd_oracle.py to
something other than itself, so that a dropped term, a wrong sign or index, or a transposed
operand fails at least one of them.  The paper prints no worked numeric example
(Figs. 1-4 are images), so there is no paper-value fixture; tests/golden/README.md says so.
"""
import math

import numpy as np
import pytest

import synth
from oracle import fdd_oracle as O

RNG = np.random.default_rng(20211008)


def _rand_u8(nsamps, nchans, seed=0):
    return np.random.default_rng(seed).integers(0, 256, size=(nsamps, nchans), dtype=np.uint8)


# ---------------------------------------------------------------- P1: O2 against a library
@pytest.mark.parametrize("n", [64, 1024, 8192])
def test_p1_naive_dft_is_rfft(n):
    x = RNG.standard_normal((3, n))
    ref = np.fft.rfft(x, axis=-1)
    got = O.naive_rdft(x)
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max() * math.sqrt(n)


def test_p1_padding_to_power_of_two():
    # zero pad to a power of two: 1000 -> 1024
    u8 = _rand_u8(1000, 2, 1)
    x = O.unpack(u8)
    assert x.shape == (2, 1024) and O.next_pow2(1000) == 1024 and O.next_pow2(1024) == 1024
    assert np.all(x[:, 1000:] == 0) and np.array_equal(x[:, :1000], u8.T.astype(float))
    ref = np.fft.rfft(np.pad(u8.T.astype(float), ((0, 0), (0, 24))), axis=-1)
    assert np.abs(O.naive_rdft(x) - ref).max() <= 1e-9


def test_p1_naive_inverse_is_irfft():
    n = 512
    Y = RNG.standard_normal((4, n // 2 + 1)) + 1j * RNG.standard_normal((4, n // 2 + 1))
    ref = np.fft.irfft(Y, n=n, axis=-1)            # library also drops Im of bins 0 and N/2 (S8)
    got = O.naive_irdft(Y, n, n)
    assert np.abs(got - ref).max() <= 1e-12
    # truncated output length
    assert np.abs(O.naive_irdft(Y, n, 300) - ref[:, :300]).max() <= 1e-12


# ---------------------------------------------------------------- P11: reduced-length inverse
@pytest.mark.parametrize("m", [0, 1, 3])
def test_p11_reduced_inverse_samples_a_band_limited_series(m):
    """PAPER.md:98.  A series whose spectrum stops below the new Nyquist bin M/2 is sampled
    exactly: y_m[n] = y[n 2^m] (periodic sampling theorem); the series is written as explicit
    cosines, so the expected values contain no transform at all."""
    n, M = 1024, 1024 >> m
    ks = np.array([0, 1, 5, M // 2 - 1][:4 if M // 2 - 1 > 5 else 2])
    amp = np.array([3.0, 1.5, -0.7, 2.2])[:ks.size]
    pha = np.array([0.0, 0.3, -1.1, 2.0])[:ks.size]
    t = np.arange(n)
    y = sum(a * np.cos(2 * np.pi * k * t / n + p) for a, k, p in zip(amp, ks, pha))
    Y = O.naive_rdft(y[None, :])
    got = O.naive_irdft_reduced(Y, n, n, m)[0]
    assert got.shape == (M,)
    assert np.abs(got - y[::1 << m]).max() <= 1e-11
    if m == 0:
        assert np.abs(got - O.naive_irdft(Y, n, n)[0]).max() <= 1e-12


def test_p11_reduced_inverse_is_dirichlet_lowpass_then_sampling():
    """Brute force in the time domain on a tiny random series: y_m[n] = sum_l y[l] D(n 2^m - l),
    D the periodic sinc of the kept band |k| <= M/2 (edge bins at half weight, textbook form
    sin(pi M u / N) / tan(pi u / N) / N); and the two tiers agree."""
    n, m = 64, 2
    M = n >> m
    y = RNG.standard_normal(n)
    Y = O.naive_rdft(y[None, :])
    got = O.naive_irdft_reduced(Y, n, n, m)[0]
    ref = np.zeros(M)
    for i in range(M):
        for l in range(n):
            u = (i << m) - l
            if u % n == 0:
                ker = M / n
            else:
                ker = math.sin(math.pi * M * u / n) / math.tan(math.pi * u / n) / n
            ref[i] += y[l] * ker
    assert np.abs(got - ref).max() <= 1e-12
    Yc = RNG.standard_normal((3, n // 2 + 1)) + 1j * RNG.standard_normal((3, n // 2 + 1))
    assert np.abs(O.irfft_reduced(Yc, n, 50, m) - O.naive_irdft_reduced(Yc, n, 50, m)).max() <= 1e-12
    assert O.irfft_reduced(Yc, n, 50, m).shape == (3, 13)          # ceil(50 / 4)


# ---------------------------------------------------------------- O3: delay law, Eq. 1
def test_delay_law_closed_values():
    # hand-evaluated Eq. 1: K * DM * (nu^-2 - nu0^-2) / tsamp
    d = O.delay_table(2, 1400.0, 1500.0, 64e-6, [30.0])
    expect = 4.148808e3 * 30.0 * (1400.0 ** -2 - 1500.0 ** -2) / 64e-6
    assert d.shape == (1, 2)
    assert abs(d[0, 0] - expect) < 1e-9 and d[0, 1] == 0.0
    assert abs(expect - 127.886) < 2e-3
    # config 2's one-sample step: trial i has exactly i samples at the lowest channel
    step = synth.one_sample_dm_step(1200.0, 1500.0, 64e-6)
    assert abs(step - 0.0617044703) < 1e-9
    d2 = O.delay_table(1024, 1200.0, 1500.0, 64e-6, step * np.arange(256))
    assert np.allclose(d2[:, 0], np.arange(256), atol=1e-9)
    assert np.all(np.diff(d2, axis=1) <= 0)      # delay falls with frequency
    assert O.valid_length(d2, 1 << 18) == (1 << 18) - 255    # S10 rounding trap
    # channel grid is an inclusive linspace (S3); single channel sits at f_hi
    assert np.allclose(O.channel_freqs(5, 100.0, 200.0), [100, 125, 150, 175, 200])
    assert O.channel_freqs(1, 100.0, 200.0)[0] == 200.0
    d1 = O.delay_table(64, 1400.0, 1500.0, 64e-6, 2.0 * np.arange(32))
    assert O.valid_length(d1, 8192) == 7927                  # BASELINE.json config 1


# ---------------------------------------------------------------- P2: DM = 0
def test_p2_dm0_is_channel_sum():
    u8 = _rand_u8(256, 5, 2)
    d = np.zeros((1, 5))
    y = O.fdd_naive(u8, d)
    assert np.abs(y[0] - u8.sum(axis=1)).max() <= 1e-9
    Y = O.fdd_naive(u8, d, mode="fourier")
    assert np.abs(Y[0] - np.fft.rfft(u8.astype(float).sum(axis=1))).max() <= 1e-8


# ---------------------------------------------------------------- P3: integer delays
@pytest.mark.parametrize("tier", ["naive", "fft", "rows"])
def test_p3_integer_delays_are_circular_shift_and_sum(tier):
    nsamps, nchans, ndm = 512, 7, 6
    u8 = _rand_u8(nsamps, nchans, 3)
    d = synth.integer_delay_table(5, ndm, nchans, 100)
    assert np.all(d == np.rint(d)) and d.max() > 50
    # integer-arithmetic reference: y[n] = sum_c x_c[(n + d_c) mod N]   (S1 semantics)
    ref = np.zeros((ndm, nsamps), dtype=np.int64)
    for j in range(ndm):
        for c in range(nchans):
            ref[j] += np.roll(u8[:, c].astype(np.int64), -int(d[j, c]))
    fn = {"naive": O.fdd_naive, "fft": O.fdd_fft,
          "rows": lambda a, b: O.fdd_rows(a, b, range(ndm))}[tier]
    y = fn(u8, d)
    assert np.abs(y - ref).max() <= 1e-9 * np.abs(ref).max()
    # the wrap puts samples from the START at the END: check one explicitly
    j, c = ndm - 1, 0
    only = np.zeros_like(u8); only[:, c] = u8[:, c]
    yc = O.fdd_fft(only, d)[j]
    s = int(d[j, c])
    assert np.allclose(yc[nsamps - s:], u8[:s, c], atol=1e-9)


# ---------------------------------------------------------------- P4: fractional delays
def test_p4_fractional_delay_is_periodic_sinc_interpolation():
    n, nchans = 32, 3
    u8 = _rand_u8(n, nchans, 4)
    d = np.array([[0.0, 0.0, 0.0], [3.25, 1.5, 0.0], [7.9, -2.4, 0.31]])
    y = O.fdd_naive(u8, d)
    ref = np.zeros_like(y)
    ks = np.arange(1, n // 2)
    for j in range(d.shape[0]):
        for c in range(nchans):
            for t in range(n):
                for m in range(n):
                    u = t - m + d[j, c]
                    kern = 1.0 + 2.0 * np.cos(2 * np.pi * ks * u / n).sum() \
                        + math.cos(math.pi * d[j, c]) * (-1.0) ** (t - m)
                    ref[j, t] += u8[m, c] * kern / n
    assert np.abs(y - ref).max() <= 1e-10 * np.abs(ref).max()
    # and the closed form of that kernel: sin((N-1) pi u/N) / sin(pi u/N)
    u = 0.37
    lhs = 1.0 + 2.0 * np.cos(2 * np.pi * ks * u / n).sum()
    assert abs(lhs - math.sin((n - 1) * math.pi * u / n) / math.sin(math.pi * u / n)) < 1e-12


# ---------------------------------------------------------------- P5: detection semantics
def test_p5_injected_pulse_peaks_at_its_trial():
    w = synth.workload("tiny")
    u8 = synth.make_filterbank(w)
    d = O.delay_table(w.nchans, w.f_lo, w.f_hi, w.tsamp, w.dm_list)
    y = O.fdd_fft(u8, d)
    peak = y.max(axis=1)
    assert int(np.argmax(peak)) == 15                       # DM 30 = trial 15 of step 2
    assert abs(int(np.argmax(y[15])) - 2048) <= 1           # t0 at the reference channel
    height = peak[15] - y[15].mean()
    assert 0.85 * 64 * 40 <= height <= 1.1 * 64 * 40        # ~ N_nu * amplitude
    # with the opposite phasor sign the pulse is dispersed twice over and never re-aligns
    y_wrong = O.fdd_fft(u8, -d)
    assert (y_wrong.max(axis=1) - y_wrong.mean(axis=1)).max() < 0.3 * height


# ---------------------------------------------------------------- P6: energy
def test_p6_parseval_and_unit_modulus():
    u8 = _rand_u8(128, 4, 6)
    d = np.array([[0.0, 0.0, 0.0, 0.0], [5.3, 2.2, 1.1, 0.0]])
    n = 128
    Y = O.fdd_naive(u8, d, mode="fourier")
    y = O.fdd_naive(u8, d, mode="time")
    for j in range(2):
        e_t = (y[j] ** 2).sum()
        e_f = (abs(Y[j, 0].real) ** 2 + 2 * (np.abs(Y[j, 1:n // 2]) ** 2).sum()
               + Y[j, n // 2].real ** 2) / n
        assert abs(e_t - e_f) <= 1e-12 * e_t
    # single channel: a pure phase rotation leaves amplitudes unaltered
    one = u8[:, :1]
    X = O.naive_rdft(O.unpack(one))
    Y1 = O.fdd_naive(one, np.array([[0.0], [17.77]]), mode="fourier")
    assert np.abs(np.abs(Y1[1]) - np.abs(X[0])).max() <= 1e-12 * np.abs(X).max()


# ---------------------------------------------------------------- P7: DC invariance
def test_p7_sum_over_time_is_independent_of_dm():
    u8 = _rand_u8(256, 6, 7)
    d = O.delay_table(6, 1200.0, 1500.0, 64e-6, [0.0, 3.3, 9.9, 14.2])
    y = O.fdd_naive(u8, d)
    total = float(u8.astype(np.int64).sum())
    assert np.abs(y.sum(axis=1) - total).max() <= 1e-12 * total * 10


# ---------------------------------------------------------------- P8: linearity / covariance
def test_p8_eq5_equals_eq6_and_shift_covariance():
    nsamps, nchans = 256, 5
    u8 = _rand_u8(nsamps, nchans, 8)
    d = O.delay_table(nchans, 1200.0, 1500.0, 64e-6, [0.0, 4.4, 11.0])
    y6 = O.fdd_naive(u8, d)                                        # Eq. 6: sum then invert
    X = O.naive_rdft(O.unpack(u8))
    k = np.arange(nsamps // 2 + 1)
    y5 = np.zeros_like(y6)
    for j in range(d.shape[0]):                                    # Eq. 5: invert then sum
        for c in range(nchans):
            y5[j] += O.naive_irdft(X[c] * O.phasor(k, d[j, c], nsamps), nsamps, nsamps)
    assert np.abs(y5 - y6).max() <= 1e-12 * np.abs(y6).max()
    s = 37
    y_roll = O.fdd_naive(np.roll(u8, s, axis=0), d)
    assert np.abs(y_roll - np.roll(y6, s, axis=1)).max() <= 1e-10 * np.abs(y6).max()


# ---------------------------------------------------------------- P9: phase accuracy
def test_p9_pure_tone_at_nineteen_thousand_cycles():
    # config-5 delays: up to ~3.8e4 samples, phases to ~1.9e4 cycles at k ~ N/2
    n, nchans = 1 << 19, 16
    nu = np.linspace(110.0, 190.0, nchans)
    dms = np.array([26.8, 81.91])
    d = dms[:, None] * (4.148808e3 * (nu ** -2 - 190.0 ** -2) / 491.52e-6)[None, :]
    assert d.max() > 3.7e4
    k0 = n // 2 - 1
    # X of an unquantised tone cos(2 pi k0 n / N) is (N/2) at bin k0 and 0 elsewhere
    bins = np.array([k0 - 1, k0, k0 + 1])
    X = np.zeros((nchans, 3), dtype=np.complex128); X[:, 1] = n / 2
    for fn in (O.phase_rotate_sum, O.phase_rotate_sum_c):
        Y = fn(X, d, n, bins=bins)
        # independent evaluation with exact rational phase: k0*d/N via Python Fractions
        from fractions import Fraction
        for j in range(2):
            acc = 0j
            for c in range(nchans):
                cyc = Fraction(k0) * Fraction(float(d[j, c])) / n
                fr = float(cyc - round(cyc))
                acc += (n / 2) * complex(math.cos(2 * math.pi * fr), math.sin(2 * math.pi * fr))
            assert abs(Y[j, 1] - acc) <= 1e-10 * abs(n / 2 * nchans)
            assert Y[j, 0] == 0 and Y[j, 2] == 0


# ---------------------------------------------------------------- P10: tiers agree
def test_p10_tiers_agree_on_tiny(oracle_c):
    w = synth.workload("tiny")
    u8 = synth.make_filterbank(w)
    d = O.delay_table(w.nchans, w.f_lo, w.f_hi, w.tsamp, w.dm_list)
    rows = [0, 7, 15, 31]
    y_naive = O.fdd_naive(u8, d[rows])
    y_fft = O.fdd_fft(u8, d[rows])
    y_rows = O.fdd_rows(u8, d, rows)
    scale = np.abs(y_naive).max()
    assert np.abs(y_fft - y_naive).max() <= 1e-11 * scale
    assert np.abs(y_rows - y_naive).max() <= 1e-11 * scale
    Y_naive = O.fdd_naive(u8, d[rows], mode="fourier")
    bins = [0, 1, 2, 1000, 4095, 4096]
    Yb = O.single_bins(u8, d, bins, rows=rows)
    assert np.abs(Yb - Y_naive[:, bins]).max() <= 1e-11 * np.abs(Y_naive).max()
    Y_rows = O.fdd_rows(u8, d, rows, mode="fourier")
    assert np.abs(Y_rows - Y_naive).max() <= 1e-11 * np.abs(Y_naive).max()
    # rows_from_spectrum is fdd_rows' last step (O5): from the NAIVE sums it gives the naive rows,
    # full rate and reduced length
    n = O.next_pow2(w.nsamps)
    assert np.abs(O.rows_from_spectrum(Y_naive, n, w.nsamps) - y_naive).max() <= 1e-11 * scale
    y_red = O.naive_irdft_reduced(Y_naive, n, w.nsamps, 2)
    assert np.abs(O.rows_from_spectrum(Y_naive, n, w.nsamps, "time", 2) - y_red).max() <= 1e-11 * scale
    assert np.array_equal(O.rows_from_spectrum(Y_naive, n, w.nsamps, "fourier", 2), Y_naive[:, :n // 8 + 1])


def test_c_matches_numpy(oracle_c):
    assert O._c_lib() is not None
    X = RNG.standard_normal((9, 33)) + 1j * RNG.standard_normal((9, 33))
    d = RNG.uniform(-50, 4e4, size=(4, 9))
    a = O.phase_rotate_sum(X, d, 64)
    b = O.phase_rotate_sum_c(X, d, 64)
    assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    bins = np.array([0, 5, 31, 32] + list(range(29)), dtype=np.int64)
    a = O.phase_rotate_sum(X, d, 64, bins=bins)
    b = O.phase_rotate_sum_c(X, d, 64, bins=bins)
    assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    acc = b.copy()
    O.phase_rotate_sum_c(X, d, 64, bins=bins, out=acc, accumulate=True)
    assert np.abs(acc - 2 * b).max() <= 1e-12 * np.abs(a).max()
    assert O.num_threads() >= 1


# ---------------------------------------------------------------- generator
def test_generator_is_deterministic_and_shaped():
    w = synth.workload("tiny")
    a = synth.make_filterbank(w)
    b = synth.make_filterbank(w)
    assert a.dtype == np.uint8 and a.shape == (8192, 64) and np.array_equal(a, b)
    assert abs(a.mean() - 128) < 0.5 and abs(a.std() - 16) < 0.5
    for name, shape in [("config2", (1 << 18, 1024, 256)), ("config3", (1 << 20, 1024, 1024)),
                        ("sweep", (1 << 20, 1024, 4096)), ("config5", (1 << 19, 400, 8192))]:
        ww = synth.workload(name)
        assert (ww.nsamps, ww.nchans, ww.ndm) == shape
    assert synth.workload("sweep", ndm=128).ndm == 128
    assert synth.workload("config5").mode == "fourier"
    assert abs(max(synth.workload("config5").dm_list) - 81.91) < 1e-9


# ---------------------------------------------------------------- row f1: beams
def test_beams_are_independent_and_linear(oracle_c):
    """fdd_beams adds no arithmetic: beam b equals the single-beam result; identical beams give
    identical rows; a beam at DM 0 is its own channel sum (P2 per beam); and, Eq. 7 being linear in
    the data, the spectrum of the sample-wise sum of two beams is the sum of their
    spectra - checked on inputs small enough that the sum stays in 8 bits."""
    rng = np.random.default_rng(71)
    beams = rng.integers(0, 120, (3, 512, 6), dtype=np.uint8)
    beams[2] = beams[0]
    d = O.delay_table(6, 1200.0, 1500.0, 64e-6, [0.0, 3.7, 11.0, 40.0])
    Y = O.fdd_beams(beams, d, mode="fourier")
    y = O.fdd_beams(beams, d, mode="time")
    assert Y.shape == (3, 4, 257) and y.shape == (3, 4, 512)
    for b in range(3):
        assert np.abs(y[b] - O.fdd_fft(beams[b], d)).max() <= 1e-11 * np.abs(y[b]).max()
        assert np.abs(y[b][0] - beams[b].astype(np.int64).sum(axis=1)).max() <= 1e-9
    assert np.array_equal(y[0], y[2]) and not np.array_equal(y[0], y[1])
    both = (beams[0].astype(np.int64) + beams[1]).astype(np.uint8)
    Ysum = O.fdd_fft(both, d, mode="fourier")
    assert np.abs(Ysum - (Y[0] + Y[1])).max() <= 1e-10 * np.abs(Ysum).max()
