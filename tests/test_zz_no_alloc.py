"""fdd_rotate_sum_static (include/fdd.h): step a4 with its scratch in a static device array, for callers
that cannot call cudaMalloc.  Its output against the existing path's (a plan's generic a4 kernel in
FOURIER mode, fdd_execute) on the same spectra and delays, within the parity bar of tests/parity.py
(PAPER.md:64, 82), on calls in a row that share the static array.

Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test."""
import numpy as np
import pytest

import parity
import synth
from oracle import fdd_oracle as O

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


def _existing_path(F, w):
    """(plan, X device address, pitch, dc_add, delays, Y of the plan's generic kernel [ndm][nbins] c64)."""
    import torch
    u8 = synth.make_filterbank(w)
    plan = F.Plan.create(w.nchans, w.nsamps, w.tsamp, w.f_lo, w.f_hi, w.dm_list)
    plan.set_kernel(F.FDD_KERNEL_GENERIC)
    d_in = torch.from_numpy(u8).cuda()
    out = torch.empty((plan.ndm, plan.nbins, 2), dtype=torch.float32, device="cuda")
    plan.execute(d_in, out, F.FDD_MODE_FOURIER)
    torch.cuda.synchronize()
    o = out.cpu().numpy()
    x_dev, pitch, dc_removed = plan.get_spectrum()
    # bin 0 of every trial DM gets back the mean a2 removed from every channel (reading S21)
    dc_add = float(np.float32(dc_removed * w.nchans))
    return plan, x_dev, pitch, dc_add, plan.get_delays(), o[..., 0] + 1j * o[..., 1]


def _static_path(F, plan, x_dev, pitch, dc_add, delays, poison=False):
    import torch
    nfft = plan.get_info()[0]
    d_delays = torch.from_numpy(np.ascontiguousarray(delays, dtype=np.float64)).cuda()
    out = torch.full((plan.ndm, plan.nbins, 2), float("nan") if poison else 0.0, dtype=torch.float32, device="cuda")
    F.rotate_sum_static(x_dev, pitch, d_delays, plan.nchans, plan.nbins, nfft, plan.ndm, out, dc_add)
    torch.cuda.synchronize()
    o = out.cpu().numpy()
    return o[..., 0] + 1j * o[..., 1]


def test_static_scratch_entry_point_matches_the_plan_path_on_calls_in_a_row(F, oracle_c):
    # A: 40 trial DMs (5 DM tiles), 4097 bins (a ragged tail of the 128-bin CTAs); B: fewer, other delays,
    # 13 trial DMs (a ragged DM tile) - the static table still holds A's entries when B runs
    wa = synth.small_workload(4100, 64, 8192, 40, dm_step=1.5)
    wb = synth.small_workload(4101, 24, 4096, 13, dm_step=0.7)
    a = _existing_path(F, wa)
    b = _existing_path(F, wb)
    try:
        for rnd, (plan, x_dev, pitch, dc_add, delays, ref) in enumerate((a, b, a, b)):
            got = _static_path(F, plan, x_dev, pitch, dc_add, delays, poison=True)
            assert np.isfinite(got.view(np.float64)).all(), f"call {rnd}: output rows not written"
            worst = parity.assert_rows(got, ref, "fourier", f"static scratch, call {rnd}")
            if rnd < 2:
                # ... and against the oracle itself (Eq. 4 + 7), the bar of every parity test
                w = (wa, wb)[rnd]
                rows = list(range(plan.ndm))
                exact = O.fdd_rows(synth.make_filterbank(w), O.delay_table(w.nchans, w.f_lo, w.f_hi, w.tsamp,
                                                                         w.dm_list), rows, mode="fourier")
                parity.assert_rows(got, exact, "fourier", f"static scratch against the oracle, call {rnd}")
            # the same 64-bit phase table on both sides (the plan's kernel walks the bins by a recurrence,
            # this one makes a fresh phasor per element): measured 3e-7, far inside the bar
            assert worst["rel_l2"] <= 1e-5, (rnd, worst)
            print("static call", rnd, plan.ndm, plan.nchans, worst)
    finally:
        a[0].destroy()
        b[0].destroy()


def test_static_scratch_entry_point_rejects_what_does_not_fit(F):
    import torch
    x = torch.zeros((4, 64, 2), dtype=torch.float32, device="cuda")
    d = torch.zeros((8, 4), dtype=torch.float64, device="cuda")
    out = torch.zeros((8, 33, 2), dtype=torch.float32, device="cuda")
    F.rotate_sum_static(x, 64, d, 4, 33, 64, 8, out)                       # fits
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0
    # nchans * round_up(ndm, 8) beyond FDD_STATIC_MAX_PHASES: a clear error, nothing launched
    nchans = 1024
    ndm = F.FDD_STATIC_MAX_PHASES // nchans + 1
    with pytest.raises(F.FddError) as e:
        F.rotate_sum_static(x, 64, d, nchans, 33, 64, ndm, out)
    assert e.value.status == F.FDD_ERR_TOO_LARGE
    assert "static scratch" in str(e.value)
    with pytest.raises(F.FddError):
        F.rotate_sum_static(x, 16, d, 4, 33, 64, 8, out)                   # pitch shorter than the rows
    with pytest.raises(F.FddError):
        F.rotate_sum_static(x, 64, d, 4, 34, 64, 8, out)                   # more bins than nfft / 2 + 1
