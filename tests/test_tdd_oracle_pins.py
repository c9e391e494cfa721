"""Pins for the time-domain comparator's oracle (oracle/tdd_oracle.py, Eq. 2)."""
import numpy as np

import synth
from oracle import fdd_oracle as O
from oracle import tdd_oracle as T


def _rand_u8(nsamps, nchans, seed):
    return np.random.default_rng(seed).integers(0, 256, size=(nsamps, nchans), dtype=np.uint8)


def test_t1_loops_and_rolls_agree_and_dm0_is_the_channel_sum():
    u8 = _rand_u8(96, 5, 1)
    d = np.array([[0, 0, 0, 0, 0], [7.2, 5.5, 3.49, 1.5, 0.0], [40.0, 30.6, 20.4, 9.5, 0.0]])
    a, b = T.tdd_loops(u8, d), T.tdd_rows(u8, d)
    assert a.dtype == np.int64 and np.array_equal(a, b)
    assert np.array_equal(a[0], u8.astype(np.int64).sum(axis=1))
    assert np.array_equal(T.tdd_rows(u8, d, rows=[2]), b[2:3])


def test_t2_rounding_is_to_the_nearest_sample_ties_up():
    """Eq. 2: "rounded to the nearest time sample".  A single channel holding a ramp makes the
    applied shift readable from the output."""
    n = 64
    u8 = np.arange(n, dtype=np.uint8).reshape(n, 1)
    for d, s in ((0.49, 0), (0.5, 1), (1.49, 1), (2.5, 3), (7.0, 7)):
        y = T.tdd_rows(u8, np.array([[d]]))[0]
        assert y[0] == s and y[n - 1] == (n - 1 + s) % n


def test_t3_integer_delays_equal_the_fourier_domain_result():
    """with the right phasors the Fourier-domain result is the time-domain one; for
    integer delays and a power-of-two length that holds sample for sample (both wrap around)."""
    u8 = _rand_u8(1024, 12, 3)
    d = synth.integer_delay_table(5, 9, 12, 300)
    ref = O.fdd_fft(u8, d)                           # the FDD oracle, fp64
    got = T.tdd_rows(u8, d)
    assert np.abs(got - ref).max() <= 1e-9 * np.abs(ref).max()


def test_t4_injected_pulse_peaks_at_its_trial():
    w = synth.workload("tiny")
    u8 = synth.make_filterbank(w)
    d = O.delay_table(w.nchans, w.f_lo, w.f_hi, w.tsamp, w.dm_list)
    y = T.tdd_rows(u8, d)
    peak = y.max(axis=1)
    assert int(np.argmax(peak)) == 15 and abs(int(np.argmax(y[15])) - 2048) <= 1
