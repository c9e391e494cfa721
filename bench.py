#!/usr/bin/env python
"""bench.py -- dedispersion rate of the FDD hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--ndm D] [--impl reference]

A step is one pass of the whole hot path (a2 unpack+transpose, a3 R2C, a4 phase-rotate-and-sum,
a5 C2R) over one seeded synthetic filterbank (synth/filterbank.py).  Default workload: the
configuration BASELINE.json's target is quoted on, config 4 at 4096 trial DMs (1024 channels x
2^20 samples), which fits one GPU.  metric = DM-trials x samples / s.

  value      K steps through fdd_execute with the input resident in HBM, CUDA events on the
             launching stream, barrier + synchronize on both sides, max over ranks
  e2e        the same metric through fdd_execute_host: pinned HOST input and output, both
             copies inside the timed region
  roofline   the dominant kernel (a4): algorithmic 8 flop per (dm, channel, bin) element over
             its mean launch duration (CUDA events recorded by the library between the stages,
             inside the timed region), against the FP32 FMA rate measured live on the same GPU
             by a register-resident FFMA2 loop
  cpu_baseline  the CPU oracle as it stands, timed on the host cores on a bounded sample

N > 1: weak scaling by trial-DM range -- every rank dedisperses the same input over its own
block of ndm trial DMs (rank r: trials r*ndm .. (r+1)*ndm - 1); no data-path collective
(DESIGN.md "Multi-GPU").  One process per GPU: under torchrun the ranks are already there; a
plain `python bench.py --gpus N` starts them itself (torch.distributed.run on 127.0.0.1) and
fails if fewer than N GPUs are visible.  --impl reference times the oracle (rank 0 only).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "dedispersion_rate"
UNIT = "DM-trials*samples/s"
FLOP_PER_ELEMENT = 8.0          # one complex MAC per (dm, channel, bin): SURVEY.md 8d


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="config4",
                    choices=["tiny", "config2", "config3", "config4", "config5", "paper"])
    ap.add_argument("--ndm", type=int, default=None, help="trial DMs (config 4 sweep point)")
    ap.add_argument("--kernel", default="auto",
                    choices=["auto", "generic", "symmetric", "symmetric2", "tensor"])
    ap.add_argument("--decimate", type=int, default=0, metavar="M",
                    help="row f3: reduced-length inverse transform, output down-sampled by 2^M "
                         "(PAPER.md:98); the rate still counts the INPUT samples dedispersed")
    ap.add_argument("--with-tdd", action="store_true",
                    help="row f4: also time the time-domain comparator (fdd_tdd_execute) on the "
                         "same input and report it as tdd_comparator")
    ap.add_argument("--beams", type=int, default=1, metavar="B",
                    help="row f1: B beams per step through fdd_execute_beams (beam 0 = the workload's "
                         "input, the others seeded noise made on the device); the rate counts all beams")
    ap.add_argument("--inverse", default="auto", choices=["auto", "cufft", "two_pass"],
                    help="step a5: the plan's choice (default), cuFFT, or the hand-written two-pass inverse")
    ap.add_argument("--y-budget-gib", type=float, default=0.0, metavar="G",
                    help="fdd_plan_set_y_budget: TIME-mode Y scratch per DM chunk (0 = the library's default)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-rows", type=int, default=3, help="DM rows the oracle sample computes")
    return ap.parse_args()


def dist_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def make_workload(args, rank: int, world: int):
    """The synthetic workload of this rank: rank r takes trial DMs [r*ndm, (r+1)*ndm)."""
    import synth
    w = synth.workload(args.workload, ndm=args.ndm)
    ndm = w.ndm
    if world > 1:
        step = w.dm_list[1] - w.dm_list[0] if ndm > 1 else 0.0
        dms = tuple(w.dm_list[0] + step * (rank * ndm + i) for i in range(ndm))
        import dataclasses
        w = dataclasses.replace(w, dm_list=dms)
    return w


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    REASONS = {
        0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap",
        0x8: "hw_slowdown", 0x10: "sync_boost", 0x20: "sw_thermal_slowdown",
        0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting",
    }

    def __init__(self, index: int, period_s: float = 0.02):
        self.samples, self.reason_bits, self.power = [], 0, []
        self.sm_max = None
        self._stop = threading.Event()
        self._thread = None
        self.period = period_s
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.reason_bits |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.nv is not None:
            self._stop.clear()
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self):
        if self._thread is not None:
            self._stop.set()
            self._thread.join()
            self._thread = None

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": 0}
        reasons = [n for b, n in self.REASONS.items() if self.reason_bits & b and n != "gpu_idle"]
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.sm_max,
                "reasons": reasons, "samples": len(self.samples),
                "power_w_max": max(self.power) if self.power else None}


# ----------------------------------------------------------------------------- CPU oracle legs
def oracle_sample(w, u8, nrows: int, cfft: int = 256):
    """Time the oracle (oracle/, as it stands) on a bounded sample of workload ``w``.

    The oracle's cost is  t_fft (O1+O2, once per input)  +  rows * t_row (O4+O5 per trial DM),
    exactly linear in the rows; both parts are measured on this box and the whole-workload time
    is t_fft + ndm * t_row.  Returns (rate, description, threads, seconds spent).
    """
    from oracle import build as obuild
    obuild.build()
    from oracle import fdd_oracle as O
    t_start = time.time()
    d = O.delay_table(w.nchans, w.f_lo, w.f_hi, w.tsamp, w.dm_list)
    n = O.next_pow2(w.nsamps)
    rng = np.random.default_rng(w.seed)
    rows = sorted({0, w.ndm - 1} | set(int(r) for r in rng.integers(0, w.ndm, max(nrows - 2, 0))))
    rows = rows[:max(nrows, 1)]
    # O1+O2 on a bounded subset of channels (cost is linear in channels), scaled to all of them
    cfft = min(w.nchans, cfft)
    t0 = time.time()
    X = np.fft.rfft(O.unpack(u8[:, :cfft], n), axis=-1)
    t_fft = (time.time() - t0) * (w.nchans / cfft)
    # O4 for the sampled rows over a bounded channel subset, scaled; O5 per row
    t0 = time.time()
    Y = O.phase_rotate_sum_c(X, d[rows][:, :cfft], n)
    t_o4 = (time.time() - t0) * (w.nchans / cfft) / len(rows)
    t_o5 = 0.0
    if w.mode == "time":
        t0 = time.time()
        np.fft.irfft(Y, n=n, axis=-1)
        t_o5 = (time.time() - t0) / len(rows)
    t_full = t_fft + w.ndm * (t_o4 + t_o5)
    rate = w.ndm * w.nsamps / t_full
    what = (f"{len(rows)} of {w.ndm} DM rows x {cfft} of {w.nchans} channels x all {w.nsamps} samples "
            f"(fp64 FFT {t_fft:.1f} s per input + {t_o4 + t_o5:.2f} s per DM row, both linear, "
            f"scaled to the whole workload: {t_full:.0f} s)")
    return rate, what, O.num_threads(), time.time() - t_start


def cpu_model() -> str:
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.lower().startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def naive_tiny_sample():
    """the NAIVE oracle (O(N^2) transforms, fdd_naive) end to end on the
    whole Tiny config (64 channels x 8192 samples x 32 trial DMs), with one thread and with all the
    threads numpy's BLAS takes on this box."""
    import synth
    from oracle import fdd_oracle as O
    w = synth.workload("tiny")
    u8 = synth.make_filterbank(w)
    d = O.delay_table(w.nchans, w.f_lo, w.f_hi, w.tsamp, w.dm_list)
    out = {"workload": "config 1 (tiny), all 32 trial DMs, naive O(N^2) DFTs", "unit": UNIT}
    try:
        from threadpoolctl import threadpool_limits
    except Exception:
        threadpool_limits = None
    if threadpool_limits is not None:
        with threadpool_limits(limits=1):
            t0 = time.time()
            O.fdd_naive(u8, d, mode="time")
            t1 = time.time() - t0
        out["single_thread_s"] = t1
        out["single_thread_value"] = w.ndm * w.nsamps / t1
    t0 = time.time()
    O.fdd_naive(u8, d, mode="time")
    ta = time.time() - t0
    out["all_cores_s"] = ta
    out["all_cores_value"] = w.ndm * w.nsamps / ta
    out["host_cores"] = os.cpu_count()
    return out


def run_reference(args, rank: int, world: int):
    """--impl reference: the oracle timed on the host cores, rank 0 only."""
    if rank != 0:
        return
    import synth
    w = make_workload(args, 0, 1)
    u8 = synth.make_filterbank(w)
    budget = 150.0 / max(args.steps + args.warmup, 1)        # seconds of CPU work per step
    rates, what, threads = [], "", 1
    nrows, cfft = 2, 256
    for it in range(args.warmup + args.steps):
        rate, what, threads, spent = oracle_sample(w, u8, nrows, cfft)
        if it >= args.warmup:
            rates.append(rate)
        if spent > budget and cfft > 16:
            cfft //= 2
    value = float(np.mean(rates))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * w.ndm * w.nsamps / value, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, 1),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": what, "host_cores": os.cpu_count(), "cpu_model": cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def kernel_source_hash() -> str:
    """sha256 (first 16 hex) over the CUDA sources without // comments and blank lines: ties static
    profile numbers to a source state."""
    import glob
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2110_03482_b200", "csrc")
    for f in sorted(glob.glob(os.path.join(csrc, "*.cu")) + glob.glob(os.path.join(csrc, "*.cuh"))):
        h.update(os.path.basename(f).encode())
        for ln in open(f, "r", errors="replace"):              # code only: comments do not stale a profile
            code = ln.split("//", 1)[0].strip()
            if code:
                h.update(code.encode())
    return h.hexdigest()[:16]


def workload_config(w, world: int):
    return {"workload": f"{w.name}: {w.nchans} channels {w.f_lo:g}-{w.f_hi:g} MHz, "
                        f"{w.nsamps} samples of {w.tsamp * 1e6:g} us, {w.ndm} trial DMs per GPU, "
                        f"{w.mode}-domain output",
            "nchans": w.nchans, "nsamps": w.nsamps, "ndm_per_gpu": w.ndm, "ndm_total": w.ndm * world,
            "mode": w.mode, "seed": w.seed,
            "l2": "inputs larger than L2 (no flush needed): u8 input, X and Y are each >= 1 GiB"
                  if w.nsamps * w.nchans > (1 << 28) else "L2 flushed between steps"}


# ----------------------------------------------------------------------------- the CUDA arm
def run_b200(args, rank: int, local_rank: int, world: int):
    import torch
    import torch.distributed as dist
    import synth
    from paper_2110_03482_b200 import build as fbuild
    if rank == 0:
        fbuild.build()
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the FDD path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    import paper_2110_03482_b200 as F
    F.load_library()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = make_workload(args, rank, world)
    u8 = synth.make_filterbank(w)                       # same bytes on every rank (same seed)
    mode = F.FDD_MODE_TIME if w.mode == "time" else F.FDD_MODE_FOURIER
    plan = F.Plan.create(w.nchans, w.nsamps, w.tsamp, w.f_lo, w.f_hi, w.dm_list)
    plan.set_kernel({"auto": F.FDD_KERNEL_AUTO, "generic": F.FDD_KERNEL_GENERIC,
                     "symmetric": F.FDD_KERNEL_SYMMETRIC,
                     "symmetric2": F.FDD_KERNEL_SYMMETRIC2,
                     "tensor": F.FDD_KERNEL_TENSOR}[args.kernel])
    nfft, nbins, valid, maxd, scratch, kernel = plan.get_info()
    if args.decimate:
        plan.set_decimation(args.decimate)
    if args.y_budget_gib > 0:
        plan.set_y_budget(int(args.y_budget_gib * (1 << 30)))
    if args.inverse != "auto":
        plan.set_inverse(F.FDD_INVERSE_TWO_PASS if args.inverse == "two_pass" else F.FDD_INVERSE_CUFFT)
    ns_out, nbins = plan.output_shape()                   # = (nsamps, nbins) at full rate
    nfft_out = nfft >> args.decimate
    d_in = torch.from_numpy(u8).cuda()
    nbeams = max(1, args.beams)
    if nbeams > 1:
        beams = torch.empty((nbeams, w.nsamps, w.nchans), dtype=torch.uint8, device="cuda")
        beams[0] = d_in
        gen = torch.Generator(device="cuda").manual_seed(w.seed + 99)
        for b in range(1, nbeams):
            beams[b] = (torch.randn((w.nsamps, w.nchans), generator=gen, device="cuda") * 16 + 128
                        ).round().clamp(0, 255).to(torch.uint8)
        d_in = beams
    lead = (nbeams,) if nbeams > 1 else ()
    if mode == F.FDD_MODE_TIME:
        out = torch.empty(lead + (w.ndm, ns_out), dtype=torch.float32, device="cuda")
    else:
        out = torch.empty(lead + (w.ndm, nbins, 2), dtype=torch.float32, device="cuda")
    flush = None
    if w.nsamps * w.nchans <= (1 << 28):
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step():
        if flush is not None:
            flush.fill_(1)
        if nbeams > 1:
            plan.execute_beams(d_in, out, nbeams, mode, stream)
        else:
            plan.execute(d_in, out, mode, stream)

    # FP32 FMA rate of this GPU, measured with the library's FFMA2 probe (~0.25 s, sustained)
    peak_tf, peak_ms = F.measure_fp32_peak(True, 1 << 19)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(torch.cuda.current_device() if "CUDA_VISIBLE_DEVICES" not in os.environ
                           else int(os.environ["CUDA_VISIBLE_DEVICES"].split(",")[local_rank]))
    plan.set_profiling(True)                              # zeroes the stage totals
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    sampler.stop()
    ms_total = ev0.elapsed_time(ev1)
    stage_ms, launches = plan.get_stage_ms()
    # (a TIME-mode plan whose Y chunks are short falls back to the FP32 kernel at its first execute:
    #  report the kernel that ran, and the scratch it holds now)
    scratch, kernel = plan.get_info()[4:6]
    own_inverse = mode == F.FDD_MODE_TIME and plan.get_inverse() == F.FDD_INVERSE_TWO_PASS
    plan.set_profiling(False)
    if flush is not None:                                  # the flush is not part of the path
        ms_total = sum(stage_ms.values())
    t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
    per_rank_ms = [ms_total / args.steps]
    if world > 1:
        allt = [torch.zeros_like(t) for _ in range(world)]
        dist.all_gather(allt, t)
        per_rank_ms = [float(x.item()) / args.steps for x in allt]
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item()) / args.steps
    units = float(w.ndm) * w.nsamps * world * nbeams      # DM-trials x samples, all ranks (and beams)
    value = units / (ms_step * 1e-3)

    # ---- the time-domain comparator on the same input (row f4; not part of `value`) -----
    tdd = None
    if args.with_tdd and mode == F.FDD_MODE_TIME and not args.decimate:
        for _ in range(2):
            plan.tdd_execute(d_in, out, stream)
        torch.cuda.synchronize()
        plan.set_profiling(True)
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record(stream)
        for _ in range(args.steps):
            plan.tdd_execute(d_in, out, stream)
        t1.record(stream)
        torch.cuda.synchronize()
        tms = t0.elapsed_time(t1) / args.steps
        st, _ = plan.get_stage_ms()
        plan.set_profiling(False)
        tdd = {"what": "time-domain shift-and-add (Eq. 2) on the same input, same GPU: "
                       "fdd_tdd_execute = u8 transpose + integer shift-and-add",
               "ms_per_step": tms, "value": float(w.ndm) * w.nsamps / (tms * 1e-3), "unit": UNIT,
               "stage_ms_per_step": {"tdd_transpose": st["tdd_transpose"] / args.steps,
                                     "tdd_shift_add": st["tdd_shift_add"] / args.steps},
               "fdd_over_tdd_time": ms_step / tms}

    # ---- end to end through the host-buffer entry point ---------------------------------
    e2e = None
    if not args.no_e2e and nbeams == 1:
        host_memory = "pinned"
        try:
            h_in = torch.from_numpy(u8).pin_memory()
            h_out = torch.empty(out.shape, dtype=torch.float32, pin_memory=True)
        except RuntimeError:                               # not enough lockable host memory
            host_memory = "pageable"
            h_in = torch.from_numpy(u8)
            h_out = torch.empty(out.shape, dtype=torch.float32)
        plan.execute_host(h_in, h_out, mode, stream)       # warm-up: staging buffers, page faults
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            plan.execute_host(h_in, h_out, mode, stream)   # returns when the result is on the host
        barrier()
        t_e2e = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(t_e2e, op=dist.ReduceOp.MAX)
        # the host link's own rate for pinned copies of this size class, measured here, so the
        # reader can see how close e2e is to the link limit (its time is mostly the copy back)
        pcie = None
        if host_memory == "pinned":
            nprobe = min(h_out.numel(), 1 << 28)                     # <= 1 GiB of floats
            hv, dv = h_out.view(-1)[:nprobe], out.view(-1)[:nprobe]
            ea, eb, ec = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            dv_keep = dv.clone()
            hv.copy_(dv, non_blocking=True)                          # warm-up
            torch.cuda.synchronize()
            ea.record(stream)
            hv.copy_(dv, non_blocking=True)
            eb.record(stream)
            dv.copy_(hv, non_blocking=True)
            ec.record(stream)
            torch.cuda.synchronize()
            dv.copy_(dv_keep)
            del dv_keep
            d2h = nprobe * 4e-9 / (ea.elapsed_time(eb) * 1e-3)
            h2d = nprobe * 4e-9 / (eb.elapsed_time(ec) * 1e-3)
            t_step = float(t_e2e.item()) / args.e2e_steps
            pcie = {"d2h_gbs_pinned_copy": d2h, "h2d_gbs_pinned_copy": h2d,
                    "probe_bytes": nprobe * 4,
                    "e2e_d2h_gbs": int(h_out.numel()) * 4e-9 / t_step,
                    "e2e_time_over_copy_floor": t_step / (int(h_out.numel()) * 4e-9 / d2h
                                                         + int(h_in.numel()) * 1e-9 / h2d)}
        e2e = {"value": units / (float(t_e2e.item()) / args.e2e_steps), "unit": UNIT, "pcie": pcie,
               "h2d_bytes_per_step": int(h_in.numel()) * world,
               "d2h_bytes_per_step": int(h_out.numel()) * 4 * world,
               "steps": args.e2e_steps, "host_memory": host_memory,
               "timer": "host perf_counter around fdd_execute_host (synchronous), max over ranks"}
        del h_in, h_out

    if rank != 0:
        plan.destroy()
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (a4) ---------------------------------------------
    # achieved = the FP32 FMA work the kernel EXECUTES (2 flop per FMA lane) over its mean launch
    # duration, against the FP32 FMA rate measured live on this GPU: a fraction of the pipe's peak,
    # always <= 1.  The symmetric kernels execute fewer FMAs per (dm, channel, bin) element than the 8
    # flop of one complex MAC (paired rows, shared three-term recurrence), so the rate at which they
    # retire the rotate-then-MAC model's work is reported beside it, not as a fraction of peak.
    elements = float(w.ndm) * w.nchans * nbins
    sum_ms = stage_ms["rotate_sum"] / args.steps
    ntl = (w.ndm + 31) // 32
    ns3 = ((ntl + 2) // 3) * 294 <= ((ntl + 1) // 2) * 232          # the library's rule (sym2_shape)
    kname, fma_lanes = {
        F.FDD_KERNEL_SYMMETRIC2: ("k_rotate_sum_sym2<%d>" % (3 if ns3 else 2),
                                  111 * 2 / 96.0 if ns3 else 79 * 2 / 64.0),
        F.FDD_KERNEL_MIXED: ("k_rotate_sum_sym2 + k_rotate_sum_krec (mixed)", 111 * 2 / 96.0),
        F.FDD_KERNEL_SYMMETRIC: ("k_rotate_sum_sym", 47 * 2 / 32.0),
        F.FDD_KERNEL_TENSOR: ("k_rotate_sum_tc", 0.0),
        # bin-recurrence kernel: 4 FMA for the MAC + 4 for the advance on 7 of 8 bins
        F.FDD_KERNEL_GENERIC: ("k_rotate_sum_krec", 7.5) if nfft <= (1 << 23)
        else ("k_rotate_sum_generic", 4.0)}[kernel]
    executed = 2.0 * fma_lanes * elements / (sum_ms * 1e-3) * 1e-12
    src_hash = kernel_source_hash()
    traffic, traffic_src, traffic_hash = None, None, None
    tpath = os.path.join(ROOT, "profiles", "roofline_traffic.csv")   # from the committed ncu summaries
    if os.path.exists(tpath) and not args.decimate:
        key = f"{w.name}/{w.ndm}/kernel{kernel}"
        for ln in open(tpath):
            f = ln.strip().split(",")
            if len(f) >= 3 and f[0] == key:
                traffic, traffic_src = float(f[1]), f[2]
                traffic_hash = f[3] if len(f) > 3 else None
    roofline = {
        "kernel": kname,
        "bound": "alu", "achieved": executed, "peak": peak_tf, "unit": "TFLOP/s",
        "frac": executed / peak_tf, "traffic": traffic,
        "traffic_source": None if traffic is None else
        f"static: profiles/{traffic_src} (one ncu --set full capture, not this run)",
        "traffic_stale": None if traffic is None else (traffic_hash != src_hash),
        "kernel_sources_sha": src_hash,
        "peak_source": "measured live: fdd_measure_fp32_peak (FFMA2 register loop, all SMs, "
                       f"{peak_ms:.0f} ms); cross-check 148 SM x 128 lanes x 2 x 1.965 GHz = 74.45",
        "achieved_is": "executed FP32 FMA lanes x 2 flop / mean launch duration (CUDA events "
                       "around the stage, inside the timed region)",
        "executed_fma_lanes_per_element": fma_lanes,
        "executed_fma_lanes_source": "static: FFMA2 counted in the SASS of the channel loop "
                                     "(profiles/*_ncu_full_*.md instruction mix), not a counter of this run",
        "algorithmic_equiv_tflops": FLOP_PER_ELEMENT * elements / (sum_ms * 1e-3) * 1e-12,
        "algorithmic_equiv_is": "8 flop (one complex MAC) per (dm, channel, bin) element / time: the "
                                "rate at which a rotate-then-MAC kernel would have to run to match; "
                                "not a fraction of peak (this kernel executes fewer flop per element)",
        "ms_per_launch": sum_ms, "share_of_step": sum_ms / ms_step,
    }
    if kernel == F.FDD_KERNEL_TENSOR:
        # tensor-core kernel: the work it executes is the tcgen05.mma stream - per launch (<= 4096
        # trial DMs), Fourier bin (in units of 4) and 64-channel stage: 3 products (hi.hi, hi.lo,
        # lo.hi) x 4 K-steps of a 128 x 64 x 16 fp16 MMA - against the measured dense bf16/fp16
        # tensor peak of this pool's B200s (sustained figure: the kernel runs inside a long step)
        try:
            pk = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pk = {}
        tpeak = pk.get("bf16_tflops_sustained", 1400.0)
        if nbeams > 1:
            grp = 4 if w.ndm <= 1024 else (2 if w.ndm <= 2048 else 1)
            nlaunch = -(-nbeams // grp) * (-(-w.ndm // 4096) if grp == 1 else 1)
        else:
            nlaunch = -(-w.ndm // 4096)
        kpad = -(-w.nchans // 64) * 64
        bpad = -(-nbins // 4) * 4
        # a one-beam launch of <= 2048 trial DMs takes 64 operand rows (UMMA M = 64: half the flop of the
        # 128-row form in the same tensor-pipe time - the pipe's peak is then out of reach by design)
        mrows = 64 if (nbeams == 1 and w.ndm <= 2048 and os.environ.get("FDD_TC_FEW") != "0") else 128
        mma_flop = nlaunch * 3.0 * 2.0 * mrows * 64 * kpad * bpad
        roofline.update({
            "bound": "tensor", "achieved": mma_flop / (sum_ms * 1e-3) * 1e-12, "peak": tpeak,
            "frac": mma_flop / (sum_ms * 1e-3) * 1e-12 / tpeak,
            "peak_source": ("MEASURED_PEAKS.json bf16_tflops_sustained (cuBLAS bf16 GEMM, seconds-long "
                            "loop; fp16 and bf16 share the kind::f16 rate); burst figure "
                            f"{pk.get('bf16_tflops')}") if pk else
                           "fallback 1.4 PFLOP/s sustained (B200_PROFILING.md): MEASURED_PEAKS.json absent",
            "achieved_is": f"executed tcgen05.mma flop (3 fp16 products of {mrows} x 64 x N_nu per bin and "
                           "launch) / mean launch duration (CUDA events around the stage)",
            "fp32_peak_tflops_measured": peak_tf,
            "algorithmic_equiv_over_fp32_peak": FLOP_PER_ELEMENT * elements / (sum_ms * 1e-3) * 1e-12 / peak_tf,
        })
        roofline.pop("executed_fma_lanes_per_element", None)
        roofline.pop("executed_fma_lanes_source", None)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": dict(workload_config(w, world), decimation_log2=args.decimate, beams=nbeams),
        "ms_per_step_per_rank": per_rank_ms,
        "tdd_comparator": tdd,
        "clocks": sampler.summary(),
        "e2e": e2e,
        # (step a5 runs this repo's own two-pass inverse or cuFFT: fdd_plan_get_inverse says which)
        "gpu_launches": int(launches["unpack"] + launches["rotate_sum"] + (launches["c2r"] if own_inverse else 0)),
        "library_calls": int(launches["r2c"] + (0 if own_inverse else launches["c2r"])),
        "inverse": ("two_pass" if own_inverse else "cufft") if mode == F.FDD_MODE_TIME else None,
        "stage_ms_per_step": {k: v / args.steps for k, v in stage_ms.items()
                              if not k.startswith("tdd_")},
        "roofline": roofline,
        "plan": {"nfft": nfft, "nbins": nbins, "valid_len": valid, "max_delay_samples": maxd,
                 "scratch_bytes": scratch, "kernel": kernel,
                 "rotate_sum_chunks_per_step": launches["rotate_sum"] / args.steps,
                 "device_free_bytes": torch.cuda.mem_get_info()[0]},
    }
    # HBM-bound stages: achieved GB/s against the measured copy bandwidth
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm = peaks.get("hbm_gbs", 6650.0)
    pitch = 2 * ((nbins + 15) // 16 * 16)
    stage_bytes = {
        "unpack": w.nchans * w.nsamps + 4.0 * w.nchans * nfft,
        "r2c": 4.0 * w.nchans * nfft + 8.0 * w.nchans * (nfft // 2 + 1),
        "c2r": (8.0 * w.ndm * nbins + 4.0 * w.ndm * nfft_out) if mode == F.FDD_MODE_TIME else 0.0,
    }
    line["hbm_stages"] = {
        k: {"algorithmic_gb": b * 1e-9, "gbs": b * 1e-9 / (line["stage_ms_per_step"][k] * 1e-3),
            "frac_of_copy_peak": b * 1e-9 / (line["stage_ms_per_step"][k] * 1e-3) / hbm}
        for k, b in stage_bytes.items() if line["stage_ms_per_step"][k] > 0}
    line["hbm_peak_gbs"] = hbm
    line["hbm_peak_source"] = "MEASURED_PEAKS.json" if peaks else "fallback 6650 (B200_PROFILING.md)"

    if nbeams > 1:
        line["beams"] = {"nbeams": nbeams, "ms_per_beam": ms_step / nbeams,
                         "rotate_sum_ms_per_beam": stage_ms["rotate_sum"] / args.steps / nbeams,
                         "what": "fdd_execute_beams: groups of 4 beams (2 above 1024 trial DMs) share one "
                                 "tensor-core a4 launch (PAPER.md:274)"}
    if world == 1 and not args.no_cpu_baseline:
        plan.destroy()
        del d_in, out
        torch.cuda.empty_cache()
        rate, what, threads, _ = oracle_sample(w, u8, args.cpu_rows)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
                                "sample": what, "host_cores": os.cpu_count(),
                                "cpu_model": cpu_model(), "naive_tiny": naive_tiny_sample()}
    else:
        plan.destroy()
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    rank, local_rank, world = dist_env()
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if world != args.gpus and world > 1:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}")
    if args.gpus > 1 and world == 1:
        # not under torchrun: start one process per GPU ourselves (same launch the driver uses)
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            raise SystemExit(f"--gpus {args.gpus} but only {have} CUDA device(s) are visible")
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
               f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    run_b200(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
