"""GPU parity: the CUDA path through the C ABI against the CPU oracle, element by element.

Tolerances are those of BASELINE.json north_star under the strict (mean-subtracted) reading,
see tests/parity.py.  Integer work (the unpack stage, integer-delay shift-and-sum rounded to
integers) is compared exactly.  Inputs are seeded and synthetic (synth/filterbank.py).
"""
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


def _run(F, plan, u8, mode):
    import torch
    d_in = torch.from_numpy(u8).cuda()
    if mode == "time":
        out = torch.empty((plan.ndm, plan.nsamps), dtype=torch.float32, device="cuda")
        plan.execute(d_in, out, F.FDD_MODE_TIME)
        torch.cuda.synchronize()
        return out.cpu().numpy()
    out = torch.empty((plan.ndm, plan.nbins, 2), dtype=torch.float32, device="cuda")
    plan.execute(d_in, out, F.FDD_MODE_FOURIER)
    torch.cuda.synchronize()
    o = out.cpu().numpy()
    return o[..., 0] + 1j * o[..., 1]


def _plan_for(F, w):
    return F.Plan.create(w.nchans, w.nsamps, w.tsamp, w.f_lo, w.f_hi, w.dm_list)


def _delays_for(w):
    return O.delay_table(w.nchans, w.f_lo, w.f_hi, w.tsamp, w.dm_list)


KERNELS = ["generic", "symmetric", "auto"]


def _set_kernel(F, plan, which):
    """auto = the fastest kernel the delay table allows (on uniform DM grids SYMMETRIC2 below 640
    trial DMs, TENSOR from there).  Returns the kernel the plan resolved to (enum fdd_kernel)."""
    plan.set_kernel({"generic": F.FDD_KERNEL_GENERIC, "symmetric": F.FDD_KERNEL_SYMMETRIC,
                     "symmetric2": F.FDD_KERNEL_SYMMETRIC2, "tensor": F.FDD_KERNEL_TENSOR,
                     "auto": F.FDD_KERNEL_AUTO}[which])
    return plan.get_info()[5]


# ------------------------------------------------------------------ stages a2 + a3
@pytest.mark.parametrize("nchans,nsamps", [(64, 8192), (7, 1000), (1, 64), (130, 4100)])
def test_unpack_and_r2c_against_fp64_rfft(F, nchans, nsamps):
    import torch
    u8 = np.random.default_rng(nchans * 7 + nsamps).integers(0, 256, (nsamps, nchans), dtype=np.uint8)
    with F.Plan.create(nchans, nsamps, 64e-6, 1200.0, 1500.0, [0.0]) as plan:
        d_in = torch.from_numpy(u8).cuda()
        out = torch.empty((1, plan.nsamps), dtype=torch.float32, device="cuda")
        plan.execute(d_in, out, F.FDD_MODE_TIME)
        torch.cuda.synchronize()
        ptr, pitch, dc_removed = plan.get_spectrum()
        assert dc_removed == 128.0 * nsamps
        assert plan.nfft == O.next_pow2(nsamps) and plan.nbins == plan.nfft // 2 + 1
        # view the plan's X in place through the CUDA array interface
        class _View:
            __cuda_array_interface__ = {"shape": (nchans, pitch, 2), "typestr": "<f4",
                                        "data": (ptr, False), "version": 2}
        xs = torch.as_tensor(_View(), device="cuda")
        X = xs.cpu().numpy()
        X = (X[..., 0] + 1j * X[..., 1])[:, :plan.nbins]
        X[:, 0] += dc_removed                      # the mean a2 takes out of the fp32 FFT
        ref = np.fft.rfft(O.unpack(u8, plan.nfft), axis=-1)
        kx = plan.get_padding()                    # zero padded: the mean is a rectangle, whose spectrum
        assert kx == (0 if nsamps == plan.nfft else min(plan.nbins, 4096))   # is missing below bin kx
        if kx:
            rect = np.zeros(plan.nfft); rect[:nsamps] = 128.0
            ref[:, 1:kx] -= np.fft.rfft(rect)[1:kx]
        # fp32 FFT of u8 data: error relative to the rms of the non-DC bins
        rms = np.sqrt((np.abs(ref[:, 1:]) ** 2).mean())
        assert np.abs(X - ref)[:, 1:].max() <= 2e-5 * rms * np.sqrt(np.log2(plan.nfft))
        assert np.abs(X[:, 0] - ref[:, 0]).max() <= 1e-6 * np.abs(ref[:, 0]).max()
        # DM = 0 output is the plain channel sum: integers, exact after rounding (a2 is exact)
        y = out.cpu().numpy()[0]
        assert np.array_equal(np.rint(y).astype(np.int64), u8.astype(np.int64).sum(axis=1))


# ------------------------------------------------------------------ config 1, whole path
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("mode", ["time", "fourier"])
def test_tiny_all_rows_against_naive_oracle(F, mode, kernel):
    w = synth.workload("tiny")
    u8 = synth.make_filterbank(w)
    d = _delays_for(w)
    ref = O.fdd_naive(u8, d, mode=mode)
    with _plan_for(F, w) as plan:
        _set_kernel(F, plan, kernel)
        nfft, nbins, valid, maxd, scratch, k = plan.get_info()
        assert (nfft, nbins, valid) == (8192, 4097, 7927) and abs(maxd - d.max()) < 1e-9
        assert np.abs(plan.get_delays() - d).max() <= 1e-9
        got = _run(F, plan, u8, mode)
    worst = parity.assert_rows(got, ref, mode, f"tiny/{mode}/{kernel}")
    print("tiny", mode, kernel, worst)
    if mode == "time":
        peak = got.max(axis=1)
        assert int(np.argmax(peak)) == 15 and abs(int(np.argmax(got[15])) - 2048) <= 1


# ------------------------------------------------------------------ ragged / edge shapes
RAGGED = [
    # nchans, nsamps, ndm, dm_step, dm0
    (5, 1000, 3, 7.5, 0.0),          # zero padding 1000 -> 1024, odd channel count
    (1, 256, 4, 10.0, 0.0),          # single channel: all delays zero
    (64, 2048, 1, 3.0, 12.0),        # single DM
    (33, 4096, 37, 1.25, -5.0),      # negative DMs, ndm ragged against every tile size
    (96, 6000, 70, 0.9, 3.3),        # padded 6000 -> 8192, two DM tiles + tail
    (2, 2, 2, 1.0, 0.0),             # smallest legal nsamps
    (1100, 512, 40, 0.5, 0.0),       # more channels than one shared-memory table chunk (1024)
    (40, 1024, 129, 0.25, 1.0),      # five 32-DM tiles: a 96-DM group + a one-row tail tile
]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("mode", ["time", "fourier"])
@pytest.mark.parametrize("nchans,nsamps,ndm,step,dm0", RAGGED)
def test_ragged_shapes(F, nchans, nsamps, ndm, step, dm0, mode, kernel):
    w = synth.small_workload(100 + nchans, nchans, nsamps, ndm, dm_step=step, dm0=dm0, mode=mode)
    u8 = synth.make_filterbank(w)
    d = _delays_for(w)
    ref = O.fdd_fft(u8, d, mode=mode)
    with _plan_for(F, w) as plan:
        _set_kernel(F, plan, kernel)
        got = _run(F, plan, u8, mode)
        assert plan.get_info()[2] == max(0, O.valid_length(d, nsamps))   # (the library clamps at 0)
    if nsamps >= 256:
        parity.assert_rows(got, ref, mode, f"ragged {nchans}x{nsamps}x{ndm}/{mode}/{kernel}")
    else:
        scale = np.abs(ref).max()
        assert np.abs(got - ref).max() <= 1e-5 * scale


@pytest.mark.parametrize("log2n,kernel", [(22, "symmetric"), (22, "auto"), (22, "generic"),
                                          (24, "auto"), (24, "generic")])
def test_long_series_phase_variants(F, oracle_c, log2n, kernel):
    """k_rotate_sum_sym2 forms its phases on the FP64 pipe with a reduced scale for
    2^21 < nfft <= 2^23 and by integer multiplies beyond; k_rotate_sum_sym always by integers;
    FDD_KERNEL_GENERIC is the bin-recurrence kernel up to 2^23 points and the SFU kernel beyond."""
    w = synth.small_workload(321, 4, 1 << log2n, 70, dm_step=0.5, dm0=0.0)
    u8 = synth.make_filterbank(w)
    d = _delays_for(w)
    rows = [0, 1, 15, 16, 31, 32, 63, 64, 69]
    ref = O.fdd_rows(u8, d, rows, mode="time")
    with _plan_for(F, w) as plan:
        _set_kernel(F, plan, kernel)
        got = _run(F, plan, u8, "time")[rows]
    parity.assert_rows(got, ref, "time", f"nfft 2^{log2n}/{kernel}")


# ------------------------------------------------------------------ row f3: reduced-length inverse
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("nsamps,m", [(8192, 1), (8192, 3), (6000, 2)])
def test_decimated_outputs_against_the_reduced_inverse_oracle(F, oracle_c, nsamps, m, kernel):
    """fdd_plan_set_decimation: TIME rows = reduced-length inverse transform,
    FOURIER rows = the first bins of the full spectrum; m = 0 afterwards restores full rate."""
    import torch
    w = synth.small_workload(500 + m, 48, nsamps, 100, dm_step=0.8)
    u8 = synth.make_filterbank(w)
    d = _delays_for(w)
    rows = list(range(w.ndm))
    ref_t = O.fdd_rows(u8, d, rows, mode="time", log2_factor=m)
    ref_f = O.fdd_rows(u8, d, rows, mode="fourier", log2_factor=m)
    d_in = torch.from_numpy(u8).cuda()
    with _plan_for(F, w) as plan:
        _set_kernel(F, plan, kernel)
        plan.set_decimation(m)
        ns_out, nb_out = plan.output_shape()
        assert ns_out == -(-nsamps // (1 << m)) and nb_out == (plan.nfft >> m) // 2 + 1
        assert ref_t.shape == (w.ndm, ns_out) and ref_f.shape == (w.ndm, nb_out)
        out_t = torch.full((w.ndm, ns_out), float("nan"), dtype=torch.float32, device="cuda")
        out_f = torch.full((w.ndm, nb_out, 2), float("nan"), dtype=torch.float32, device="cuda")
        plan.execute(d_in, out_t, F.FDD_MODE_TIME)
        plan.execute(d_in, out_f, F.FDD_MODE_FOURIER)
        torch.cuda.synchronize()
        got_t = out_t.cpu().numpy()
        o = out_f.cpu().numpy()
        got_f = o[..., 0] + 1j * o[..., 1]
        parity.assert_rows(got_t, ref_t, "time", f"decimated 2^{m}/{kernel}")
        parity.assert_rows(got_f, ref_f, "fourier", f"decimated 2^{m}/{kernel}")
        plan.set_decimation(0)
        full = _run(F, plan, u8, "time")
    parity.assert_rows(full, O.fdd_rows(u8, d, rows, mode="time"), "time", "full rate again")
    with pytest.raises(F.FddError):
        with _plan_for(F, w) as plan:
            plan.set_decimation(40)


def test_non_uniform_dm_list_and_kdm_override(F):
    rng = np.random.default_rng(5)
    dms = np.sort(rng.uniform(0, 300, size=45))
    dms[7] = dms[6]                                      # duplicate (S20)
    w = synth.small_workload(77, 48, 4096, 2)
    u8 = synth.make_filterbank(w)
    kdm = 1.0 / 2.41e-4                                  # the paper's constant
    d = O.delay_table(48, w.f_lo, w.f_hi, w.tsamp, dms, k_dm=kdm)
    ref = O.fdd_fft(u8, d)
    with F.Plan.create(48, 4096, w.tsamp, w.f_lo, w.f_hi, dms) as plan:
        plan.set_kdm(kdm)
        assert np.abs(plan.get_delays() - d).max() <= 1e-9
        got = _run(F, plan, u8, "time")
    parity.assert_rows(got, ref, "time", "non-uniform DM list")


def test_kernel_selection_follows_the_dm_grid(F):
    """AUTO: SYMMETRIC2 on a uniform grid AND on a piecewise-uniform DM plan whose step changes
    between 32-DM tiles (its CTA groups end where the step changes), GENERIC otherwise; each
    against the fp64 oracle, the piecewise plan also through the 32-DM-tile kernel."""
    w = synth.small_workload(78, 40, 2048, 2)
    u8 = synth.make_filterbank(w)
    uniform = np.arange(96) * 0.75
    piecewise = np.concatenate([np.arange(32) * 0.5, 16.0 + np.arange(64) * 1.0,
                                80.0 + np.arange(96) * 2.0, 272.0 + np.arange(20) * 4.0])
    random = np.sort(np.random.default_rng(6).uniform(0, 80, size=70))
    for dms, want in ((uniform, F.FDD_KERNEL_SYMMETRIC2), (piecewise, F.FDD_KERNEL_SYMMETRIC2),
                      (random, F.FDD_KERNEL_GENERIC)):
        d = O.delay_table(40, w.f_lo, w.f_hi, w.tsamp, dms)
        for mode in ("time", "fourier"):
            ref = O.fdd_fft(u8, d, mode=mode)
            with F.Plan.create(40, 2048, w.tsamp, w.f_lo, w.f_hi, dms) as plan:
                assert plan.get_info()[5] == want
                if want == F.FDD_KERNEL_GENERIC:
                    with pytest.raises(F.FddError):
                        plan.set_kernel(F.FDD_KERNEL_SYMMETRIC2)
                got = _run(F, plan, u8, mode)
                parity.assert_rows(got, ref, mode, f"kernel selection {want}/{mode}")
                if dms is piecewise:
                    plan.set_kernel(F.FDD_KERNEL_SYMMETRIC)
                    parity.assert_rows(_run(F, plan, u8, mode), ref, mode, "piecewise/32-DM tiles")


def test_dm_plan_with_step_changes_inside_tiles_runs_mixed(F):
    """A search-style DM plan (three ranges, each with its own step, lengths not multiples of 32):
    AUTO = MIXED - the tiles that hold a step change take the generic kernel, the rest the
    shared-recurrence one; against the fp64 oracle, both modes, and bit-compared with the generic
    kernel on the rows of a generic tile."""
    w = synth.small_workload(79, 40, 4096, 2)
    u8 = synth.make_filterbank(w)
    dms = np.concatenate([np.arange(50) * 0.5, 25.0 + np.arange(70) * 1.0, 95.0 + np.arange(45) * 2.0])
    d = O.delay_table(40, w.f_lo, w.f_hi, w.tsamp, dms)
    for mode in ("time", "fourier"):
        ref = O.fdd_fft(u8, d, mode=mode)
        with F.Plan.create(40, 4096, w.tsamp, w.f_lo, w.f_hi, dms) as plan:
            assert plan.get_info()[5] == F.FDD_KERNEL_MIXED
            with pytest.raises(F.FddError):
                plan.set_kernel(F.FDD_KERNEL_SYMMETRIC2)
            got = _run(F, plan, u8, mode)
            parity.assert_rows(got, ref, mode, f"mixed/{mode}")
            plan.set_kernel(F.FDD_KERNEL_GENERIC)
            gen = _run(F, plan, u8, mode)
            # trials 32..63 hold the first step change (at trial 50): generic in both runs
            assert np.array_equal(got[32:64], gen[32:64])
            assert not np.array_equal(got[0:32], gen[0:32])
    rnd = np.sort(np.random.default_rng(8).uniform(0, 80, size=70))
    with F.Plan.create(40, 4096, w.tsamp, w.f_lo, w.f_hi, rnd) as plan:
        assert plan.get_info()[5] == F.FDD_KERNEL_GENERIC
        with pytest.raises(F.FddError):
            plan.set_kernel(F.FDD_KERNEL_MIXED)


# ------------------------------------------------------------------ P3 on the GPU: exact integers
def _integer_reference(u8, d, rows):
    rows = list(rows)
    ref = np.zeros((len(rows), u8.shape[0]), dtype=np.int64)
    for c in range(u8.shape[1]):
        col = u8[:, c].astype(np.int64)
        for i, j in enumerate(rows):
            ref[i] += np.roll(col, -int(d[j, c]))
    return ref


@pytest.mark.parametrize("table,kernel", [("jitter", "generic"), ("jitter", "auto"),
                                          ("progression", "symmetric"), ("progression", "symmetric2"),
                                          ("progression", "tensor"),
                                          ("progression", "auto"), ("progression", "generic")])
def test_integer_delays_equal_circular_shift_and_sum(F, table, kernel):
    """Pin P3 through every a4 kernel: whole-sample delays make the result an exact circular
    shift-and-sum, so the reference is integer arithmetic with no FFT in it ("the same
    results as with time-domain dedispersion").  "jitter": delays with no structure (bin-recurrence
    kernel); "progression": d[j][c] = j a_c with integer a_c, which the paired-row kernels take."""
    nchans, nsamps, ndm = 128, 1 << 14, 100
    u8 = np.random.default_rng(9).integers(0, 256, (nsamps, nchans), dtype=np.uint8)
    d = synth.integer_delay_table(11, ndm, nchans, 3000) if table == "jitter" else \
        synth.integer_progression_delay_table(ndm, nchans, 30)
    ref = _integer_reference(u8, d, range(ndm))
    with F.Plan.create_from_delays(nchans, nsamps, d) as plan:
        used = _set_kernel(F, plan, kernel)
        want = {"generic": F.FDD_KERNEL_GENERIC, "symmetric": F.FDD_KERNEL_SYMMETRIC,
                "symmetric2": F.FDD_KERNEL_SYMMETRIC2, "tensor": F.FDD_KERNEL_TENSOR,
                "auto": F.FDD_KERNEL_GENERIC if table == "jitter" else F.FDD_KERNEL_SYMMETRIC2}[kernel]
        assert used == want
        got = _run(F, plan, u8, "time")
        o = _run(F, plan, u8, "fourier")
    # integer sums of 128 bytes (<= 32640): fp32 path must land within 0.05 of the integer
    assert np.abs(got - ref).max() <= 0.05
    assert np.array_equal(np.rint(got).astype(np.int64), ref)
    parity.assert_rows(got, ref.astype(np.float64), "time", "integer delays")
    # FOURIER output = forward DFT of the integer rows (library rfft of exact integers)
    parity.assert_rows(o, np.fft.rfft(ref.astype(np.float64), axis=-1), "fourier", "integer delays")


# ------------------------------------------------------------------ host-buffer entry point
def test_execute_host_against_the_oracle(F):
    """fdd_execute_host (host buffers, pinned and pageable) against the fp64 oracle, and bit-equal
    to fdd_execute on device buffers."""
    import torch
    w = synth.small_workload(31, 64, 8192, 48)
    u8 = synth.make_filterbank(w)
    d = _delays_for(w)
    with _plan_for(F, w) as plan:
        h_in = torch.from_numpy(u8).pin_memory()
        h_out = torch.full((plan.ndm, plan.nsamps), float("nan"), dtype=torch.float32).pin_memory()
        plan.execute_host(h_in, h_out, F.FDD_MODE_TIME)
        parity.assert_rows(h_out.numpy(), O.fdd_fft(u8, d, mode="time"), "time", "execute_host/time")
        h_outf = torch.full((plan.ndm, plan.nbins, 2), float("nan"), dtype=torch.float32)   # pageable
        plan.execute_host(u8, h_outf, F.FDD_MODE_FOURIER)
        gotf = h_outf.numpy()[..., 0] + 1j * h_outf.numpy()[..., 1]
        parity.assert_rows(gotf, O.fdd_fft(u8, d, mode="fourier"), "fourier", "execute_host/fourier")
        assert np.array_equal(h_out.numpy(), _run(F, plan, u8, "time"))
        assert np.array_equal(gotf, _run(F, plan, u8, "fourier"))


def test_execute_host_output_ring_wraps(F):
    """More DM chunks (384 rows each) than the 3 the device-side output ring holds: every row
    against the fp64 oracle, both modes."""
    import torch
    w = synth.small_workload(32, 16, 2048, 4 * 384 + 50, dm_step=0.05)
    u8 = synth.make_filterbank(w)
    d = _delays_for(w)
    with _plan_for(F, w) as plan:
        for mode, shape in (("time", (plan.ndm, plan.nsamps)), ("fourier", (plan.ndm, plan.nbins, 2))):
            h_out = torch.full(shape, float("nan"), dtype=torch.float32).pin_memory()
            plan.execute_host(u8, h_out, F.FDD_MODE_TIME if mode == "time" else F.FDD_MODE_FOURIER)
            got = h_out.numpy()
            if mode == "fourier":
                got = got[..., 0] + 1j * got[..., 1]
            parity.assert_rows(got, O.fdd_fft(u8, d, mode=mode), mode, f"execute_host ring/{mode}")
            dev = _run(F, plan, u8, mode)
            # (not bit-equal: fdd_execute takes the tensor-core kernel at 1586 trial DMs, the 384-row
            #  chunks of the host path the FP32 kernel)
            assert np.abs(got - dev).max() <= 1e-4 * np.abs(dev).max()


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("budget_rows", [20, 32, 100, 400])
def test_dm_chunked_time_path(F, budget_rows, kernel):
    """TIME mode with a Y scratch smaller than the plan (fdd_plan_set_y_budget): a4 + a5 run chunk
    after chunk - 16-row chunks off the 32-DM tiling (generic kernel, C2R), one 32-DM tile, 96-DM
    groups, 384-row batches + a 72-row tail - through fdd_execute and fdd_execute_host."""
    import torch
    w = synth.small_workload(41, 24, 2048, 456, dm_step=0.11)        # ndm a multiple of 8
    u8 = synth.make_filterbank(w)
    ref = O.fdd_fft(u8, _delays_for(w), mode="time")
    with _plan_for(F, w) as plan:
        _set_kernel(F, plan, kernel)
        plan.set_y_budget(budget_rows * 1040 * 8)                     # rows of 1025 -> 1040 float2
        plan.prepare(F.FDD_MODE_TIME)
        got = _run(F, plan, u8, "time")
        parity.assert_rows(got, ref, "time", f"chunked {budget_rows}/{kernel}")
        h_out = torch.full((plan.ndm, plan.nsamps), float("nan"), dtype=torch.float32).pin_memory()
        plan.execute_host(u8, h_out, F.FDD_MODE_TIME)
        parity.assert_rows(h_out.numpy(), ref, "time", f"chunked host {budget_rows}/{kernel}")
        plan.set_y_budget(0)
        parity.assert_rows(_run(F, plan, u8, "time"), ref, "time", "default budget again")
        plan.set_y_budget(3 * 1040 * 8)                               # not even 8 rows
        with pytest.raises(F.FddError):
            _run(F, plan, u8, "time")


@pytest.mark.parametrize("kernel", ["auto", "generic"])
@pytest.mark.parametrize("mode", ["time", "fourier"])
def test_prepared_execute_is_captured_in_a_cuda_graph(F, mode, kernel):
    """After fdd_plan_prepare an execute allocates nothing and never synchronises (include/fdd.h):
    it can be captured in a CUDA graph, and the replay gives the oracle's rows."""
    import torch
    w = synth.small_workload(43, 32, 4096, 70, dm_step=0.4, mode=mode)
    u8 = synth.make_filterbank(w)
    ref = O.fdd_fft(u8, _delays_for(w), mode=mode)
    m = F.FDD_MODE_TIME if mode == "time" else F.FDD_MODE_FOURIER
    d_in = torch.from_numpy(u8).cuda()
    with _plan_for(F, w) as plan:
        _set_kernel(F, plan, kernel)
        shape = (plan.ndm, plan.nsamps) if mode == "time" else (plan.ndm, plan.nbins, 2)
        out = torch.zeros(shape, dtype=torch.float32, device="cuda")
        plan.prepare(m)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):                   # the first execute of this plan, under capture
            plan.execute(d_in, out, m, torch.cuda.current_stream())
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        if mode == "fourier":
            got = got[..., 0] + 1j * got[..., 1]
    parity.assert_rows(got, ref, mode, f"graph replay/{mode}/{kernel}")


def test_streams_determinism_and_plan_churn(F):
    """Executes on a non-default stream, repeated executes are bit-identical (no atomics, fixed
    summation order), and creating / destroying plans gives the device memory back."""
    import torch
    w = synth.small_workload(33, 96, 4096, 200, dm_step=0.3)
    u8 = synth.make_filterbank(w)
    d_in = torch.from_numpy(u8).cuda()
    free0 = None
    first = None
    for it in range(6):
        with _plan_for(F, w) as plan:
            out = torch.empty((plan.ndm, plan.nsamps), dtype=torch.float32, device="cuda")
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                plan.execute(d_in, out, F.FDD_MODE_TIME, st)
                plan.execute(d_in, out, F.FDD_MODE_TIME, st)
            st.synchronize()
            got = out.cpu().numpy()
            del out
        if first is None:
            first = got
        assert np.array_equal(got, first)
        torch.cuda.synchronize()
        torch.cuda.empty_cache()
        if free0 is None:                  # after the first plan: cuFFT and kernel modules are loaded
            free0 = torch.cuda.mem_get_info()[0]
    assert torch.cuda.mem_get_info()[0] >= free0 - (8 << 20)


def test_stage_profile_and_errors(F):
    import torch
    w = synth.small_workload(32, 16, 1024, 8)
    u8 = synth.make_filterbank(w)
    with _plan_for(F, w) as plan:
        plan.set_profiling(True)
        _run(F, plan, u8, "time")
        ms, launches = plan.get_stage_ms()
        assert all(v >= 0 for v in ms.values()) and ms["rotate_sum"] > 0
        assert launches["unpack"] == 1 and launches["r2c"] == 1 and launches["rotate_sum"] >= 1
        with pytest.raises(F.FddError):
            plan.execute(torch.zeros(4, device="cuda"), 0, F.FDD_MODE_TIME)     # NULL out
        with pytest.raises(F.FddError):
            plan.execute(torch.zeros(4, device="cuda"), torch.zeros(4, device="cuda"), 7)
    # delays longer than the series: nothing is valid (not a negative length)
    with F.Plan.create_from_delays(2, 64, np.array([[0.0, 0.0], [100.0, 3.0]])) as plan:
        assert plan.get_info()[2] == 0
    tf, ms_ = F.measure_fp32_peak(True, 256)
    assert tf > 1.0


# ------------------------------------------------------------------ full-size configs (sampled rows)
def _sampled_rows(ndm, n, seed):
    rng = np.random.default_rng(seed)
    rows = {0, ndm - 1}
    while len(rows) < min(n, ndm):
        rows.add(int(rng.integers(0, ndm)))
    return sorted(rows)


class _FullSize:
    """Inputs and oracle spectra of the full-size configs, made once per test session.

    Configs 3 and 4 share one input (seed 1003) and one DM step, so trial j is the same DM at
    every point of the config-4 sweep: the oracle's O1..O4 run once per distinct DM row and O5
    (O.rows_from_spectrum) once per output wanted of it."""
    u8 = {}
    Y = {}                                   # (input name, trial index) -> oracle Y row (complex128)
    sums = {}                                # input name -> (per-sample channel sums, grand total)
    dev = {}                                 # input name -> the input on the device

    @classmethod
    def channel_sums(cls, name):
        key, u8 = cls.input(name)
        if key not in cls.sums:
            cs = u8.sum(axis=1, dtype=np.int64)
            cls.sums[key] = (cs, float(cs.sum()))
        return cls.sums[key]

    @classmethod
    def device_input(cls, name):
        import torch
        key, u8 = cls.input(name)
        if key not in cls.dev:
            cls.dev.clear()                  # one resident input at a time
            cls.dev[key] = torch.from_numpy(u8).cuda()
        return cls.dev[key]

    @classmethod
    def input(cls, name):
        key = "config3" if name in ("config3", "config4", "sweep") else name
        if key not in cls.u8:
            cls.u8[key] = synth.make_filterbank(synth.workload(key))
        return key, cls.u8[key]

    @classmethod
    def spectrum_rows(cls, name, w, rows):
        key, u8 = cls.input(name)
        todo = [j for j in rows if (key, j) not in cls.Y]
        if todo:
            Y = O.fdd_rows(u8, _delays_for(w), todo, mode="fourier")
            for j, y in zip(todo, Y):
                cls.Y[(key, j)] = y
        return np.stack([cls.Y[(key, j)] for j in rows])


def _full_size_point(F, name, ndm, rows, kernel_want, decimate=0, force=None, inverse="auto"):
    """One full-size TIME execute at `ndm` trial DMs; sampled rows against the oracle."""
    import torch
    w = synth.workload(name, ndm=ndm)
    torch.cuda.empty_cache()
    _, u8 = _FullSize.input(name)
    Y = _FullSize.spectrum_rows(name, w, rows)
    ref = O.rows_from_spectrum(Y, O.next_pow2(w.nsamps), w.nsamps, "time", decimate)
    with _plan_for(F, w) as plan:
        assert plan.get_info()[2] == w.nsamps - (w.ndm - 1)
        if force:
            _set_kernel(F, plan, force)
        assert plan.get_info()[5] == kernel_want
        if decimate:
            plan.set_decimation(decimate)
        if inverse != "auto":
            plan.set_inverse(F.FDD_INVERSE_TWO_PASS if inverse == "two_pass" else F.FDD_INVERSE_CUFFT)
        ns_out, _ = plan.output_shape()
        d_in = _FullSize.device_input(name)
        out = torch.empty((plan.ndm, ns_out), dtype=torch.float32, device="cuda")
        plan.execute(d_in, out, F.FDD_MODE_TIME)
        torch.cuda.synchronize()
        got = out[rows].cpu().numpy()
        if not decimate:
            # properties that hold at any size: DM 0 is the exact channel sum; DC invariance (P7)
            y0 = out[0].cpu().numpy()
            chan_sum, total = _FullSize.channel_sums(name)
            assert np.array_equal(np.rint(y0).astype(np.int64), chan_sum)
            sums = out.double().sum(dim=1).cpu().numpy()
            assert np.abs(sums - total).max() <= 2e-6 * total
    worst = parity.assert_rows(got, ref, "time", f"{name}/{ndm}/decimate {decimate}")
    print(name, ndm, "decimate", decimate, "rows", rows, worst)
    return worst


@pytest.mark.slow
def test_full_size_config2(F, oracle_c):
    w = synth.workload("config2")
    _full_size_point(F, "config2", w.ndm, _sampled_rows(w.ndm, 16, w.seed), F.FDD_KERNEL_SYMMETRIC2)


# trials that the sweep points share (so the oracle computes each once) + every point's last row
_SWEEP_POOL = [0, 37, 101, 300, 777, 1500, 3000]


@pytest.mark.slow
@pytest.mark.parametrize("ndm", [128, 256, 512, 1024, 2048, 4096])
def test_full_size_config4_dm_sweep(F, oracle_c, ndm):
    """BASELINE.json configs[3]: every point of the DM-count sweep on the config-3 input, in the
    plan bench.py times (1024 = config 3; 4096 = the default bench workload; 128 takes the 64-DM
    group instance of the sym2 kernel, the others 96-DM groups with different tails)."""
    rows = sorted({j for j in _SWEEP_POOL if j < ndm} | {ndm - 1, ndm // 2 + 15, ndm // 2 + 16})
    # AUTO: the tensor-core kernel (+ the hand-written two-pass inverse) from 1024 trial DMs up, the
    # shared-recurrence FP32 kernel (+ cuFFT's half-length C2C) below
    _full_size_point(F, "config4", ndm, rows, F.FDD_KERNEL_TENSOR if ndm >= 1024 else F.FDD_KERNEL_SYMMETRIC2)


@pytest.mark.slow
def test_full_size_config4_tensor_kernel_cufft_inverse(F, oracle_c):
    """The tensor-core kernel followed by cuFFT's C2R (FDD_INVERSE_CUFFT), which AUTO no longer takes."""
    rows = sorted({j for j in _SWEEP_POOL if j < 1024} | {1023})
    _full_size_point(F, "config4", 1024, rows, F.FDD_KERNEL_TENSOR, inverse="cufft")


@pytest.mark.slow
@pytest.mark.parametrize("ndm", [1024, 4096])
def test_full_size_config4_fp32_kernel(F, oracle_c, ndm):
    """The same sweep points through FDD_KERNEL_SYMMETRIC2 (the FP32 CUDA-core path and its fused
    pre-twiddle + half-length inverse transform), which AUTO no longer takes at these sizes."""
    rows = sorted({j for j in _SWEEP_POOL if j < ndm} | {ndm - 1})
    _full_size_point(F, "config4", ndm, rows, F.FDD_KERNEL_SYMMETRIC2, force="symmetric2")


@pytest.mark.slow
@pytest.mark.parametrize("m,inverse", [(1, "auto"), (2, "auto"), (3, "auto"), (3, "two_pass")])
def test_full_size_config4_decimated(F, oracle_c, m, inverse):
    """Row f3 at config-4 size (512 trial DMs): reduced-length inverse transform.  The
    low-pass shrinks the rms of the series while cuFFT's fp32 error stays relative to its mean, so
    m = 3 passes with little margin; the hand-written inverse (mean added after the transform) does
    not have that dependence."""
    rows = sorted({j for j in _SWEEP_POOL if j < 512} | {511, 271, 272})
    worst = _full_size_point(F, "config4", 512, rows, F.FDD_KERNEL_SYMMETRIC2, decimate=m, inverse=inverse)
    if inverse == "two_pass":
        assert worst["rel_l2"] <= 5e-5


@pytest.mark.slow
def test_full_size_config5_fourier(F, oracle_c):
    import torch
    w = synth.workload("config5")
    u8 = synth.make_filterbank(w)
    d = _delays_for(w)
    rows = _sampled_rows(w.ndm, 6, w.seed) + [2680]           # DM 26.8 = trial 2680
    rows = sorted(set(rows))
    ref = O.fdd_rows(u8, d, rows, mode="fourier")
    bins = sorted(set(np.random.default_rng(55).integers(1, w.nsamps // 2, 62).tolist()
                      + [1, w.nsamps // 2]))
    ref_bins = O.single_bins(u8, d, bins, rows=rows)            # straight from the definition
    with _plan_for(F, w) as plan:
        d_in = torch.from_numpy(u8).cuda()
        out = torch.empty((plan.ndm, plan.nbins, 2), dtype=torch.float32, device="cuda")
        plan.execute(d_in, out, F.FDD_MODE_FOURIER)
        torch.cuda.synchronize()
        o = out[rows].cpu().numpy()
        got = o[..., 0] + 1j * o[..., 1]
        power = (out[:, 1:, 0].double() ** 2 + out[:, 1:, 1].double() ** 2)
        # the periodic pulse train (P = 0.714 s, fundamental near bin 360.9) is brightest at DM 26.8
        harm = [int(round(h * w.nsamps * w.tsamp / 0.714)) - 1 for h in range(1, 9)]
        hp = power[:, harm].sum(dim=1).cpu().numpy()
        assert abs(int(np.argmax(hp)) - 2680) <= 3
    worst = parity.assert_rows(got, ref, "fourier", "config5")
    print("config5 rows", rows, worst)
    rms = np.sqrt((np.abs(ref[:, 1:]) ** 2).mean())
    assert np.abs(got[:, bins] - ref_bins).max() <= 1e-3 * rms
    assert np.abs(ref[:, bins] - ref_bins).max() <= 1e-9 * rms     # P10 at full size


@pytest.mark.slow
def test_paper_workload_at_its_own_shape(F, oracle_c):
    """bench.py --workload paper at the paper's shape: 1024 channels x 4 687 500
    samples of 64 us zero padded to 2^23, band 1181-1581 MHz, trial DMs 0, 2, 4, ...  With padding
    the mean of the u8 data is not a single bin, so it goes through both fp32 transforms."""
    import torch
    w = synth.workload("paper", ndm=128)
    u8 = synth.make_filterbank(w)
    d = _delays_for(w)
    rows = [0, 1, 31, 64, 96, 127]
    ref = O.fdd_rows(u8, d, rows, mode="time")
    torch.cuda.empty_cache()                 # the plan holds 2 x 34 GB + cuFFT workspace: give back torch's cache
    with _plan_for(F, w) as plan:
        assert plan.nfft == 1 << 23 and plan.get_info()[5] == F.FDD_KERNEL_SYMMETRIC2
        d_in = torch.from_numpy(u8).cuda()
        out = torch.empty((plan.ndm, plan.nsamps), dtype=torch.float32, device="cuda")
        plan.execute(d_in, out, F.FDD_MODE_TIME)
        torch.cuda.synchronize()
        got = out[rows].cpu().numpy()
    worst = parity.assert_rows(got, ref, "time", "paper workload, 1024 channels")
    print("paper shape rows", rows, worst)


@pytest.mark.slow
@pytest.mark.parametrize("table", ["jitter", "progression", "progression_tensor"])
def test_full_size_integer_delays(F, table):
    """P3 at 1024 channels x 2^20 samples: no FFT anywhere in the reference.  "progression"
    (d[j][c] = j a_c, integer a_c) runs the hot kernel of the bench path, k_rotate_sum_sym2 with
    96-DM groups and the mirrored epilogue; "progression_tensor" (4096 trial DMs) the tensor-core
    kernel k_rotate_sum_tc; "jitter" the bin-recurrence kernel."""
    import torch
    nchans, nsamps = 1024, 1 << 20
    _, u8 = _FullSize.input("config3")
    if table == "jitter":
        ndm, d, want = 64, synth.integer_delay_table(13, 64, nchans, 1023), F.FDD_KERNEL_GENERIC
        rows = [0, 1, 17, 31, 32, 40, 62, 63]
    elif table == "progression":
        ndm, d, want = 192, synth.integer_progression_delay_table(192, nchans, 5), F.FDD_KERNEL_SYMMETRIC2
        rows = [0, 1, 15, 16, 31, 32, 95, 96, 111, 112, 190, 191]
    else:
        # 4096 trial DMs of one sample per trial at the bottom channel: AUTO takes the tcgen05 kernel
        ndm, d, want = 4096, synth.integer_progression_delay_table(4096, nchans, 1), F.FDD_KERNEL_TENSOR
        rows = [0, 1, 31, 32, 63, 64, 2047, 2048, 2111, 4032, 4094, 4095]
    ref = _integer_reference(u8, d, rows)
    with F.Plan.create_from_delays(nchans, nsamps, d) as plan:
        assert plan.get_info()[5] == want
        d_in = torch.from_numpy(u8).cuda()
        out = torch.empty((plan.ndm, plan.nsamps), dtype=torch.float32, device="cuda")
        plan.execute(d_in, out, F.FDD_MODE_TIME)
        torch.cuda.synchronize()
        got = out[rows].cpu().numpy()
    parity.assert_rows(got, ref.astype(np.float64), "time", f"integer delays ({table}), full size")
    # sums of 1024 bytes reach 1.3e5 where the fp32 ulp is 1/64: the rounded value is the integer
    assert np.abs(got - ref).max() <= 0.25
    assert np.array_equal(np.rint(got).astype(np.int64), ref)


# ------------------------------------------------------------------ tensor-core kernel (tcgen05)
def test_tensor_core_conventions_selftest(F):
    """fdd_tc_selftest: fp16 A[128][64] B[64][64] -> A B^T through the operand layout, descriptors,
    tcgen05.mma sequence and TMEM read-out of FDD_KERNEL_TENSOR; the reference is a numpy matmul of
    the same fp16 values in fp64 (products of fp16 values are exact in fp32: only the summation
    order differs)."""
    import torch
    rng = np.random.default_rng(17)
    a = rng.standard_normal((128, 64)).astype(np.float16)
    b = rng.standard_normal((64, 64)).astype(np.float16)
    d = torch.zeros((128, 64), dtype=torch.float32, device="cuda")
    F.tc_selftest(torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda(), d)
    torch.cuda.synchronize()
    ref = a.astype(np.float64) @ b.astype(np.float64).T
    assert np.abs(d.cpu().numpy() - ref).max() <= 2e-5 * np.abs(ref).max()


@pytest.mark.parametrize("mode", ["time", "fourier"])
@pytest.mark.parametrize("nchans,nsamps,ndm,step", [
    (64, 8192, 32, None),            # config-1 shape on a one-sample grid: half a tile
    (100, 4096, 200, 0.3),           # ragged channels (two 64-channel stages, 28 padded), 3 tiles + 8 rows
    (256, 1000, 4096, 0.02),         # all 64 tiles, padded series (1000 -> 1024), last item 1 live bin
    (1024, 2048, 300, 0.05),         # the most channels the kernel stages
    # launches of <= 32 tiles take 64 operand rows (UMMA M = 64) and share the generator warps differently
    (64, 2048, 1000, 0.05),          # 16 tiles: both 8-tile halves of the one Z warp live
    (128, 1024, 1500, 0.03),         # 24 tiles: 16-tile halves, the second one half live
    (64, 1024, 2048, 0.02),          # 32 tiles, the most of that form
    (64, 1024, 2100, 0.02),          # 33 tiles: the 128-row form again
])
def test_tensor_core_kernel_against_the_oracle(F, oracle_c, nchans, nsamps, ndm, step, mode):
    w = synth.small_workload(600 + nchans, nchans, nsamps, ndm, dm_step=step, mode=mode)
    u8 = synth.make_filterbank(w)
    d = _delays_for(w)
    rows = list(range(ndm)) if ndm <= 300 else sorted(
        set(range(0, ndm, 61)) | {31, 32, 63, 64, ndm - 1} |
        {j for j in (511, 512, 543, 1023, 1024, 1055, 1535, 1536, 2047, 2048, 2079) if j < ndm})
    ref = O.fdd_rows(u8, d, rows, mode=mode)
    with _plan_for(F, w) as plan:
        plan.set_kernel(F.FDD_KERNEL_TENSOR)
        assert plan.get_info()[5] == F.FDD_KERNEL_TENSOR
        got = _run(F, plan, u8, mode)[rows]
    worst = parity.assert_rows(got, ref, mode, f"tensor {nchans}x{nsamps}x{ndm}/{mode}")
    print("tensor", nchans, nsamps, ndm, mode, worst)


@pytest.mark.parametrize("ndm,want", [(608, "symmetric2"), (640, "tensor")])
def test_auto_takes_the_tensor_kernel_from_640_trial_dms(F, oracle_c, ndm, want):
    """AUTO on a uniform DM grid: the FP32 shared-recurrence kernel below 640 trial DMs, the
    tensor-core kernel (its 64-row form) from there - each against the oracle, TIME mode, so that the
    a5 behind either kernel is part of the check."""
    w = synth.small_workload(640 + ndm, 48, 2048, ndm, dm_step=0.04, mode="time")
    u8 = synth.make_filterbank(w)
    d = _delays_for(w)
    rows = sorted(set(range(0, ndm, 53)) | {31, 32, 511, 512, ndm - 1})
    ref = O.fdd_rows(u8, d, rows, mode="time")
    with _plan_for(F, w) as plan:
        assert plan.get_info()[5] == {"symmetric2": F.FDD_KERNEL_SYMMETRIC2, "tensor": F.FDD_KERNEL_TENSOR}[want]
        got = _run(F, plan, u8, "time")[rows]
        assert plan.get_info()[5] == {"symmetric2": F.FDD_KERNEL_SYMMETRIC2, "tensor": F.FDD_KERNEL_TENSOR}[want]
    parity.assert_rows(got, ref, "time", f"auto at {ndm} trial DMs")


# ------------------------------------------------------------------ row f1: several beams, one plan
@pytest.mark.parametrize("mode", ["time", "fourier"])
@pytest.mark.parametrize("nbeams,ndm,kernel", [
    (1, 96, "auto"),        # one beam = fdd_execute
    (4, 200, "auto"),       # one group of 4 beams sharing the pair phasors (tensor-core launch)
    (7, 1000, "auto"),      # 4 + 3 beams (the group of 3 runs as 2 + 1)
    (3, 1500, "auto"),      # 1025..2048 trial DMs: groups of 2
    (2, 70, "generic"),     # a plan that cannot share: beam after beam
])
def test_multi_beam_against_the_oracle(F, oracle_c, nbeams, ndm, kernel, mode):
    """fdd_execute_beams: every beam against the oracle's beam-by-beam definition."""
    import torch
    nchans, nsamps = 96, 2048
    ws = [synth.small_workload(900 + 7 * b, nchans, nsamps, ndm, dm_step=0.07, mode=mode) for b in range(nbeams)]
    beams = np.stack([synth.make_filterbank(w) for w in ws])
    d = _delays_for(ws[0])
    rows = list(range(ndm)) if ndm <= 200 else sorted(set(range(0, ndm, 97)) | {63, 64, ndm - 1})
    ref = O.fdd_beams(beams, d, rows, mode=mode)
    with _plan_for(F, ws[0]) as plan:
        _set_kernel(F, plan, kernel)
        shape = (nbeams, ndm, plan.nsamps) if mode == "time" else (nbeams, ndm, plan.nbins, 2)
        out = torch.full(shape, float("nan"), dtype=torch.float32, device="cuda")
        plan.execute_beams(torch.from_numpy(beams).cuda(), out, nbeams,
                           F.FDD_MODE_TIME if mode == "time" else F.FDD_MODE_FOURIER)
        torch.cuda.synchronize()
        got = out[:, rows].cpu().numpy()
        if mode == "fourier":
            got = got[..., 0] + 1j * got[..., 1]
    for b in range(nbeams):
        parity.assert_rows(got[b], ref[b], mode, f"beam {b} of {nbeams}/{ndm}/{mode}")


@pytest.mark.slow
def test_multi_beam_config3_eight_beams(F, oracle_c):
    """BASELINE.json config 3 (1024 channels x 2^20 samples x 1024 trial DMs) with 8 beams: beam 0 is
    the config-3 input, the others fresh seeded noise; two tensor-core launches of 4 beams each."""
    import torch
    w = synth.workload("config3")
    _, u8 = _FullSize.input("config3")
    nbeams = 8
    torch.cuda.empty_cache()
    d_in = torch.empty((nbeams, w.nsamps, w.nchans), dtype=torch.uint8, device="cuda")
    d_in[0] = torch.from_numpy(u8).cuda()
    gen = torch.Generator(device="cuda").manual_seed(4242)
    for b in range(1, nbeams):
        d_in[b] = (torch.randn((w.nsamps, w.nchans), generator=gen, device="cuda") * 16 + 128).round().clamp(0, 255).to(torch.uint8)
    check = {0: [0, 37, 527, 1023], 5: [1, 300, 1023]}
    with _plan_for(F, w) as plan:
        out = torch.empty((nbeams, w.ndm, w.nsamps), dtype=torch.float32, device="cuda")
        plan.execute_beams(d_in, out, nbeams, F.FDD_MODE_TIME)
        torch.cuda.synchronize()
        for b, rows in check.items():
            beam = d_in[b].cpu().numpy()
            ref = O.fdd_rows(beam, _delays_for(w), rows, mode="time")
            worst = parity.assert_rows(out[b, rows].cpu().numpy(), ref, "time", f"config 3, beam {b} of 8")
            print("config3 beams", b, rows, worst)


# ------------------------------------------------------------------ step a5: both inverse transforms
@pytest.mark.parametrize("kernel", ["auto", "symmetric", "tensor"])
@pytest.mark.parametrize("nchans,nsamps,ndm,step", [
    (64, 8192, 40, 1.5),             # nfft 2^13: M = 4096 = 64 x 64
    (33, 128, 5, 0.4),               # the shortest series the hand-written inverse takes (M = 8 x 8)
    (20, 6000, 70, 0.9),             # zero padded, output cropped to 6000 of 8192 samples
    (8, 1 << 17, 33, 2.0),           # M = 2^16 = 256 x 256
    (12, 1001, 9, 0.3),              # odd series length
    (4, 1 << 14, 9, 1.1),            # M = 2^13 = 64 x 128: every transform length of the two passes once
    (4, 1 << 15, 9, 1.3),            # M = 2^14 = 128 x 128
    (4, 1 << 16, 6, 1.7),            # M = 2^15 = 128 x 256
    (4, 1 << 18, 5, 2.3),            # M = 2^17 = 256 x 512
    (4, 1 << 19, 5, 3.1),            # M = 2^18 = 512 x 512
    (3, 1 << 21, 3, 5.0),            # M = 2^20 = 1024 x 1024
    (2, 1 << 22, 3, 7.0),            # M = 2^21 = 1024 x 2048
])
def test_inverse_transform_choices(F, oracle_c, nchans, nsamps, ndm, step, kernel):
    """FDD_INVERSE_TWO_PASS (the hand-written two-pass inverse, which also restores the mean after the
    transform) and FDD_INVERSE_CUFFT (C2R, or SYMMETRIC2's fused pre-twiddle + C2C) against the oracle."""
    w = synth.small_workload(1300 + nchans, nchans, nsamps, ndm, dm_step=step)
    u8 = synth.make_filterbank(w)
    ref = O.fdd_rows(u8, _delays_for(w), range(ndm), mode="time")
    with _plan_for(F, w) as plan:
        _set_kernel(F, plan, kernel)
        for which in (F.FDD_INVERSE_AUTO, F.FDD_INVERSE_TWO_PASS, F.FDD_INVERSE_CUFFT, F.FDD_INVERSE_TWO_PASS):
            plan.set_inverse(which)
            got = _run(F, plan, u8, "time")
            if which != F.FDD_INVERSE_AUTO:
                # (every length here is one the hand-written inverse takes)
                assert plan.get_inverse() == which
            else:
                # AUTO: cuFFT's half-length C2C behind SYMMETRIC2's fused pre-twiddle (not for zero-padded
                # series, whose a4 writes plain sums), the hand-written inverse behind every other kernel
                fused = plan.get_info()[5] == F.FDD_KERNEL_SYMMETRIC2 and nsamps & (nsamps - 1) == 0
                assert plan.get_inverse() == (F.FDD_INVERSE_CUFFT if fused else F.FDD_INVERSE_TWO_PASS)
            worst = parity.assert_rows(got, ref, "time", f"inverse {which}/{kernel}/{nchans}x{nsamps}")
            print("inverse", which, kernel, nchans, nsamps, worst)
        with pytest.raises(F.FddError):
            plan.set_inverse(7)


def test_in_place_forward_transform(F, oracle_c, monkeypatch):
    """Plans whose unpacked copy alone would take 16 GiB (the paper's 2^23-point series) unpack into the
    spectra buffer and transform in place; FDD_R2C_INPLACE forces that layout at a test size, through
    fdd_execute, fdd_execute_host and fdd_execute_beams."""
    import torch
    monkeypatch.setenv("FDD_R2C_INPLACE", "1")
    w = synth.small_workload(77, 40, 3000, 70, dm_step=0.6)
    u8 = synth.make_filterbank(w)
    ref = O.fdd_rows(u8, _delays_for(w), range(w.ndm), mode="time")
    with _plan_for(F, w) as plan:
        parity.assert_rows(_run(F, plan, u8, "time"), ref, "time", "in-place R2C")
        h_out = torch.empty((plan.ndm, plan.nsamps), dtype=torch.float32).pin_memory()
        plan.execute_host(u8, h_out, F.FDD_MODE_TIME)
        parity.assert_rows(h_out.numpy(), ref, "time", "in-place R2C, host")
        beams = np.stack([u8, u8[::-1].copy()])
        out = torch.empty((2, plan.ndm, plan.nsamps), dtype=torch.float32, device="cuda")
        plan.execute_beams(torch.from_numpy(beams).cuda(), out, 2, F.FDD_MODE_TIME)
        torch.cuda.synchronize()
        parity.assert_rows(out[0].cpu().numpy(), ref, "time", "in-place R2C, beams")
