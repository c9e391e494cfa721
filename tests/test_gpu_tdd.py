"""Row f4: the time-domain comparator (fdd_tdd_execute) against its integer oracle -- bit exact."""
import numpy as np
import pytest

import synth
from oracle import fdd_oracle as O
from oracle import tdd_oracle as T

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2110_03482_b200 import build as fbuild
    fbuild.build()
    import paper_2110_03482_b200 as pkg
    pkg.load_library()
    return pkg


def _tdd(F, w, u8, d=None):
    import torch
    d_in = torch.from_numpy(u8).cuda()
    if d is None:
        plan = F.Plan.create(w.nchans, w.nsamps, w.tsamp, w.f_lo, w.f_hi, w.dm_list)
    else:
        plan = F.Plan.create_from_delays(u8.shape[1], u8.shape[0], d)
    with plan:
        out = torch.full((plan.ndm, plan.nsamps), float("nan"), dtype=torch.float32, device="cuda")
        plan.tdd_execute(d_in, out)
        torch.cuda.synchronize()
        return out.cpu().numpy(), _oracle_delays(w, d)


def _oracle_delays(w, d=None, rows=None):
    """The ORACLE's delay table (never the product's), checked to hold no rounding tie in the rows
    compared: Eq. 2 rounds to the nearest sample, and an entry within 1e-6 of a half-integer could
    legitimately round either way on the two sides.  (Config 3 has true ties: channel 868 sits at
    16000/11 MHz, where the one-sample DM step gives exactly 32.5 samples at trial 288.)"""
    if d is None:
        d = O.delay_table(w.nchans, w.f_lo, w.f_hi, w.tsamp, w.dm_list)
    d = np.asarray(d, dtype=np.float64)
    sel = d if rows is None else d[list(rows)]
    frac = sel - np.floor(sel)
    assert np.abs(frac - 0.5).min() > 1e-6, "a delay sits on a rounding tie: pick other rows"
    return d


def test_tiny_all_rows_and_the_pulse(F):
    w = synth.workload("tiny")
    u8 = synth.make_filterbank(w)
    got, d = _tdd(F, w, u8)
    ref = T.tdd_rows(u8, d)
    assert np.array_equal(got.astype(np.int64), ref) and np.array_equal(got, ref.astype(np.float32))
    assert int(np.argmax(got.max(axis=1))) == 15


@pytest.mark.parametrize("nchans,nsamps,ndm,step,dm0", [
    (5, 1000, 3, 7.5, 0.0),          # odd channel count, length not a multiple of 64
    (1, 256, 4, 10.0, 0.0),          # single channel
    (33, 4100, 37, 1.25, -5.0),      # negative DMs (shifts wrap backwards), ragged everything
    (300, 3001, 70, 0.9, 3.3),       # more channels than one 16-bit accumulation run (256)
    (2, 2, 2, 1.0, 0.0),             # smallest legal nsamps: every shift wraps
])
def test_ragged_shapes_bit_exact(F, nchans, nsamps, ndm, step, dm0):
    w = synth.small_workload(200 + nchans, nchans, nsamps, ndm, dm_step=step, dm0=dm0)
    u8 = synth.make_filterbank(w)
    got, d = _tdd(F, w, u8)
    assert np.array_equal(got.astype(np.int64), T.tdd_rows(u8, d))


def test_saturated_input_does_not_overflow_the_packed_sums(F):
    u8 = np.full((2048, 700), 255, dtype=np.uint8)
    d = synth.integer_delay_table(3, 40, 700, 500)
    got, _ = _tdd(F, None, u8, d)
    assert np.all(got == 255.0 * 700)


@pytest.mark.slow
def test_config3_sampled_rows_and_agreement_with_fdd(F):
    """Full size: sampled rows bit exact; and for rows whose delays are all integers (DM 0 and
    the channel pattern of the one-sample step does not give more) the FDD output agrees."""
    import torch
    w = synth.workload("config3")
    u8 = synth.make_filterbank(w)
    rows = [0, 1, 31, 32, 500, 1023]
    with F.Plan.create(w.nchans, w.nsamps, w.tsamp, w.f_lo, w.f_hi, w.dm_list) as plan:
        d_in = torch.from_numpy(u8).cuda()
        out = torch.empty((plan.ndm, plan.nsamps), dtype=torch.float32, device="cuda")
        plan.tdd_execute(d_in, out)
        torch.cuda.synchronize()
        got = out[rows].cpu().numpy()
        d = _oracle_delays(w, rows=rows)
        out_f = torch.empty_like(out)
        plan.execute(d_in, out_f, F.FDD_MODE_TIME)
        torch.cuda.synchronize()
        fdd0 = out_f[0].cpu().numpy()
    assert np.array_equal(got.astype(np.int64), T.tdd_rows(u8, d, rows))
    assert np.array_equal(np.rint(fdd0).astype(np.int64), got[0].astype(np.int64))
