/* fdd.h -- C ABI of the B200-native Fourier-domain dedispersion (FDD) hot path.
 *
 * Method: Bassa, Romein, Veenboer, van der Vlugt & Wijnholds, "Fourier-domain dedispersion",
 * arXiv:2110.03482.  Citations "PAPER.md:<line>" refer to the paper text the build was given.
 *
 * One fdd_execute() call runs, on one GPU and one CUDA stream, with no host synchronisation once
 * the plan has been prepared for that mode (fdd_plan_prepare; an unprepared plan does the same
 * allocations inside its first execute, which may then synchronise the device):
 *
 *   a2  unpack + transpose (+ zero pad)   u8 [nsamps][nchans] -> f32 [nchans][nfft]
 *                                          (Algorithm 1 lines 10-11)
 *   a3  batched real-to-complex FFT        X[c][k] = sum_n x[c][n] e^{-2 pi i k n / nfft}
 *                                          (Eq. 3; cuFFT)
 *   a4  phase-rotate-and-sum               Y[j][k] = sum_c X[c][k] e^{+2 pi i k d[j][c] / nfft}
 *                                          (Eq. 4 + Eq. 7; the hot kernel)
 *   a5  TIME:    batched inverse real FFT and 1/nfft scaling (Eq. 6; cuFFT: a
 *                half-length complex transform of the pre-twiddled spectrum a4 writes, or C2R)
 *       FOURIER: nothing -- Y is the output (periodicity searches)
 *
 * with the delay table (a1, Eq. 1, against the highest channel)
 *
 *   d[j][c] = k_dm * dm_j * (nu_c^-2 - f_hi^-2) / tsamp   [samples],
 *   nu_c    = f_lo + c (f_hi - f_lo) / (nchans - 1)       [MHz]   (nu_0 = f_hi if nchans == 1)
 *
 * built once per plan on the host in long double.  nfft is the next power of two >= nsamps
 * (PAPER.md:155).  Sign convention: y_j[n] = sum_c x_c[(n + d[j][c]) mod nfft] (band-limited
 * for fractional d), i.e. dispersed pulses are re-aligned at the arrival time of the highest
 * channel; with the forward kernel e^{-2 pi i k n / nfft} of Eq. 3 that is the phasor
 * e^{+2 pi i k d / nfft}.  (Eq. 4's literal minus sign belongs to the opposite transform
 * sign; the two give conjugate spectra and identical time series.  DESIGN.md, reading S1.)
 *
 * Conventions
 *   - All pointers named "host" are host memory, all named "dev"/in_u8/out (fdd_execute) are
 *     DEVICE memory of the current CUDA device.  The caller owns in_u8 and out; the plan owns
 *     every table, scratch buffer, cuFFT plan and workspace.  in_u8 is never modified.
 *   - A plan belongs to the device that was current at creation and is not re-entrant: at most
 *     one execute in flight per plan.  Different plans may run concurrently.  Results are
 *     deterministic: the same plan and input give the same bits on every execute.
 *   - Every function returns FDD_OK (0) or a negative fdd_status; nothing throws, nothing
 *     prints, no global state.  A failed create leaves *plan_out = NULL and frees everything.
 *   - There is no CPU fallback: without a CUDA device fdd_plan_create returns FDD_ERR_CUDA.
 */
#ifndef FDD_H_
#define FDD_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fdd_plan fdd_plan;   /* opaque */

enum fdd_mode {
    FDD_MODE_TIME = 0,      /* out = float32 [ndm][nsamps], includes the 1/nfft of Eq. 6          */
    FDD_MODE_FOURIER = 1    /* out = float2  [ndm][nfft/2+1] (re, im), unnormalised Y of Eq. 7    */
};

enum fdd_status {
    FDD_OK = 0,
    FDD_ERR_INVALID_ARG = -1,
    FDD_ERR_ALLOC = -2,
    FDD_ERR_CUDA = -3,
    FDD_ERR_CUFFT = -4,
    FDD_ERR_UNSUPPORTED = -5,
    FDD_ERR_TOO_LARGE = -6     /* fdd_rotate_sum_static: the problem does not fit the static scratch */
};

/* Kernel choice for step a4 (fdd_plan_set_kernel). */
enum fdd_kernel {
    FDD_KERNEL_AUTO = 0,       /* symmetric kernel where the DM grid allows it, else generic     */
    FDD_KERNEL_GENERIC = 1,    /* any delay table: phasors by recurrence along the bins from an
                                  exactly range-reduced seed per (channel, DM, 8 bins)           */
    FDD_KERNEL_SYMMETRIC = 2,  /* DM tiles in arithmetic progression: paired +-m rows */
    FDD_KERNEL_SYMMETRIC2 = 3, /* same, up to three adjacent 32-DM tiles per CTA sharing one phasor
                                  recurrence; the groups follow the uniform segments of the DM
                                  plan (a group ends where the DM step changes)                  */
    FDD_KERNEL_MIXED = 4,      /* SYMMETRIC2 for the 32-DM tiles that are arithmetic progressions,
                                  GENERIC for the few that are not (a DM plan whose step changes
                                  inside a tile)                                                */
    FDD_KERNEL_TENSOR = 5      /* uniform DM grids (ONE arithmetic progression over all trial DMs),
                                  <= 1024 channels, nfft <= 2^23: per Fourier bin the sum is a real
                                  matrix product over the channels (tile-centre rotated spectra x
                                  pair phasors), run on the tcgen05 tensor cores with fp16 hi + lo
                                  operands and fp32 accumulation in TMEM           */
};

/* Step a5 (fdd_plan_set_inverse). */
enum fdd_inverse {
    FDD_INVERSE_CUFFT = 0,     /* cuFFT: C2R, or the half-length C2C fed by SYMMETRIC2's fused pre-twiddle  */
    FDD_INVERSE_TWO_PASS = 1,  /* the hand-written two-pass inverse real transform, nfft = 2^7 .. 2^23
                                  (radix-8 butterflies in registers): forms the half-length spectrum in
                                  its first pass and adds the series' mean after the transform, so fp32
                                  works on a series of rms sigma instead of 256 sigma (TIME-mode error
                                  about 2x smaller).  Faster than cuFFT's C2R (18.8 vs 21.1 ms at 4096 x
                                  2^20, 55 vs 82 ms at 1024 x 2^23), slower than the C2C behind
                                  SYMMETRIC2's fused pre-twiddle; cuFFT for other lengths              */
    FDD_INVERSE_AUTO = 2       /* the default: TWO_PASS where it applies, a4 writes plain sums (every a4
                                  kernel but SYMMETRIC2) and its 512 MiB intermediate fits; CUFFT
                                  otherwise                                                            */
};

/* Stage indices for fdd_plan_get_stage_ms. */
enum fdd_stage {
    FDD_STAGE_UNPACK = 0, FDD_STAGE_R2C = 1, FDD_STAGE_ROTATE_SUM = 2, FDD_STAGE_C2R = 3,
    FDD_STAGE_TDD_TRANSPOSE = 4, FDD_STAGE_TDD_SHIFT_ADD = 5,     /* fdd_tdd_execute only */
    FDD_NUM_STAGES = 6
};

/* a1. Create a plan for nchans channels whose centres run evenly from f_lo_mhz (channel 0) to
 * f_hi_mhz (channel nchans-1), nsamps time samples of tsamp_s seconds, and the trial DMs
 * dm_list_host[0..ndm) in pc cm^-3 (HOST pointer, copied; any finite values, any order).
 * Requires nchans >= 1, nsamps >= 2, tsamp_s > 0, 0 < f_lo_mhz <= f_hi_mhz, ndm >= 1.
 * Dispersion constant k_dm = 4.148808e3 MHz^2 pc^-1 cm^3 s (fdd_plan_set_kdm to change).
 * Allocates all device scratch (see fdd_plan_get_info for the size). */
int fdd_plan_create(fdd_plan **plan_out, int nchans, long long nsamps, double tsamp_s,
                    double f_lo_mhz, double f_hi_mhz, const double *dm_list_host, int ndm);

/* Same, from an explicit delay table delay_samples_host[ndm][nchans] (HOST, row-major, in
 * samples, any finite values) instead of frequencies and DMs.  Integer delays make the result
 * an exact circular shift-and-sum, which is how the tests pin the kernels without any FFT in
 * the reference. */
int fdd_plan_create_from_delays(fdd_plan **plan_out, int nchans, long long nsamps,
                                const double *delay_samples_host, int ndm);

/* Rebuild the delay and phase tables with another dispersion constant (Eq. 1's k_DM; the paper
 * quotes (2.41e-4)^-1 = 4149.378).  Only for plans made by fdd_plan_create. Synchronises the
 * device (it re-uploads tables the previous execute may still be reading). */
int fdd_plan_set_kdm(fdd_plan *plan, double k_dm);

/* Down-sampling by a reduced-length inverse transform ("this down-sampling can be
 * efficiently implemented by reducing the length of the inverse Fourier transform").  With
 * log2_factor = m > 0 every trial DM is formed only up to the new Nyquist bin nfft / 2^(m+1), so
 * step a4 does 2^-m of the work, and step a5 is an inverse transform of nfft / 2^m points:
 *   TIME    rows of ceil(nsamps / 2^m) floats: the ideal low-pass of the full-rate series sampled
 *           every 2^m samples, in the same units (scaled by 1 / nfft)
 *   FOURIER rows of nfft / 2^(m+1) + 1 float2: the first bins of the full spectrum
 * (fdd_plan_get_output_shape gives both lengths).  Meant for the high-DM plans of a search, where
 * dispersive smearing exceeds 2^m samples.  m = 0 restores full rate.  Requires nfft / 2^m >= 4.
 * Synchronises the device and drops the TIME-mode scratch, which the next execute re-creates. */
int fdd_plan_set_decimation(fdd_plan *plan, int log2_factor);

/* Elements per output row: TIME floats (nsamps_out) and FOURIER float2 (nbins_out).  Either pointer
 * may be NULL. */
int fdd_plan_get_output_shape(const fdd_plan *plan, long long *nsamps_out, long long *nbins_out);

/* Choose the a4 kernel (enum fdd_kernel).  FDD_ERR_UNSUPPORTED if FDD_KERNEL_SYMMETRIC is asked
 * or FDD_KERNEL_SYMMETRIC2 for a delay table that is not in arithmetic progression within every
 * 32-DM tile (tiles count from the first trial DM), or if FDD_KERNEL_TENSOR is asked for a table that
 * is not ONE progression over all trial DMs (or has more than 1024 channels, or nfft > 2^23).  AUTO
 * takes the fastest kernel the table allows: TENSOR (uniform DM grids with at least 640 trial DMs -
 * its cost is the same for any number of trial DMs of a launch up to 1024, up to 2048 and up to 4096
 * (64 or 128 operand rows); a TIME-mode plan whose sums must be processed in chunks of fewer than
 * 640 rows stays on SYMMETRIC2), else
 * SYMMETRIC2 (uniform DM grids, and piecewise-uniform DM plans whose segments are multiples
 * of 32 trial DMs), MIXED (piecewise-uniform plans with any segment lengths: only the tiles that
 * contain a step change run on the about 3.5 times slower generic kernel; at least half of the
 * tiles must be progressions), else GENERIC.  FDD_KERNEL_MIXED may be asked for whenever at least
 * one tile is a progression. */
int fdd_plan_set_kernel(fdd_plan *plan, int kernel);

/* Make everything an fdd_execute / fdd_rotate_sum_only in `mode` (enum fdd_mode) needs that the plan
 * creates lazily, so that the execute itself allocates nothing, uploads nothing and never
 * synchronises (it can then be captured in a CUDA graph):
 *   TIME     the Y scratch (up to 24 GiB, 64 GiB on FDD_KERNEL_TENSOR; see fdd_plan_set_y_budget), the inverse cuFFT plans and
 *            the shared cuFFT workspace
 *   both     the bin-recurrence tables if any trial DM runs on FDD_KERNEL_GENERIC, the launch
 *            shapes (DM-tile groups) of the shared-recurrence kernel, and the fp64 table of a
 *            zero-padded plan (fdd_plan_get_spectrum)
 * Call it again after fdd_plan_set_kernel, fdd_plan_set_kdm, fdd_plan_set_decimation or
 * fdd_plan_set_y_budget.  Synchronises the device.  Not needed for correctness: an unprepared plan
 * does the same work inside its first execute.  (The staging buffers of fdd_execute_host and the
 * tables of fdd_tdd_execute are still made on their first call.) */
int fdd_plan_prepare(fdd_plan *plan, int mode);

/* Choose the inverse transform of step a5 (enum fdd_inverse; default FDD_INVERSE_AUTO).  Synchronises the device and drops the
 * TIME-mode scratch (re-made by fdd_plan_prepare or the next TIME execute). */
int fdd_plan_set_inverse(fdd_plan *plan, int which);

/* *which = the inverse transform the plan's last TIME-mode prepare / execute used: FDD_INVERSE_TWO_PASS
 * or FDD_INVERSE_CUFFT (also before any). */
int fdd_plan_get_inverse(const fdd_plan *plan, int *which);

/* TIME mode keeps the sums Y of a chunk of trial DMs in plan-owned scratch between a4 and a5.  The
 * chunk is as many rows as fit `bytes` (default 24 GiB - 64 GiB for a plan on FDD_KERNEL_TENSOR, whose
 * cost is per launch, not per row - and never more than half of the free device memory), rounded down to whole inverse-FFT batches (384 rows), 96-DM groups, 32-DM tiles
 * or multiples of 8 rows; plans with more trial DMs run a4 + a5 chunk after chunk (the paper's
 * DM_outer batches, without re-doing a2 + a3).  bytes = 0 restores the default.
 * FDD_ERR_ALLOC from the next TIME execute / prepare if not even 8 rows fit.  Synchronises the
 * device and drops the TIME-mode scratch. */
int fdd_plan_set_y_budget(fdd_plan *plan, size_t bytes);

/* Run a2..a5 asynchronously on cuda_stream (a cudaStream_t passed as void*; NULL = legacy
 * default stream).
 *   in_u8  DEVICE, uint8 [nsamps][nchans], channel fastest, channel 0 = f_lo
 *   out    DEVICE, TIME:    float  [ndm][nsamps]; all nsamps samples of the circular result are
 *                           written, the first valid_len are free of wrap-around
 *                  FOURIER: float2 [ndm][nfft/2+1]; equals the forward DFT (kernel
 *                           e^{-2 pi i k n/nfft}) of the full-length circular TIME row times nfft/nfft,
 *                           i.e. unnormalised; bins 0 and nfft/2 keep their imaginary parts.
 * Errors: FDD_ERR_INVALID_ARG (NULL pointers, bad mode), FDD_ERR_CUDA / FDD_ERR_CUFFT with the
 * output undefined. */
int fdd_execute(fdd_plan *plan, const unsigned char *in_u8, void *out, int mode,
                void *cuda_stream);

/* End-to-end convenience for HOST buffers: copies in_host (uint8 [nsamps][nchans]) to the
 * device, runs fdd_execute, copies the result to out_host (layout as fdd_execute's out), and
 * returns after the result has landed (synchronises cuda_stream).  Pinned host memory makes
 * the copies asynchronous and overlapped with compute (TIME mode copies finished DM chunks
 * back while later chunks are still being transformed, as Algorithm 1 lines 19-22 do);
 * pageable memory works but is slower.  Staging buffers are plan-owned and
 * allocated on first use. */
int fdd_execute_host(fdd_plan *plan, const unsigned char *in_host, void *out_host, int mode,
                     void *cuda_stream);

/* Several beams (or repeated observations) of the same receiver with one plan - the paper's route to
 * sharing the phase rotations ("reusing phase rotations ... multiple beams").
 *   in_u8  DEVICE, uint8 [nbeams][nsamps][nchans], every beam laid out as for fdd_execute
 *   out    DEVICE, [nbeams] outputs of fdd_execute, one after the other
 * On a uniform DM grid with at most 2048 trial DMs and 1024 channels, groups of 4 beams (2 above 1024
 * trial DMs) run step a4 as ONE tensor-core launch: per Fourier bin the pair phasors are generated
 * once and contracted against the tile-centre-rotated spectra of all beams of the group (the beams
 * take the place of further trial-DM tiles in the rows of the matrix product, FDD_KERNEL_TENSOR), so
 * a4 costs the same for 4 beams as for 1.  Other plans run beam after beam.  Steps a2, a3 and a5 run
 * per beam.  The group's spectra (and, in TIME mode, sums) live in plan-owned scratch allocated on the
 * first call (which may synchronise the device).  Results equal nbeams separate fdd_execute calls up
 * to the kernels' rounding (the kernel choice may differ). */
int fdd_execute_beams(fdd_plan *plan, const unsigned char *in_u8, void *out, int nbeams, int mode,
                      void *cuda_stream);

/* Free everything the plan owns.  NULL is a no-op returning FDD_OK. */
int fdd_plan_destroy(fdd_plan *plan);

/* Any output pointer may be NULL.  valid_len = nsamps - ceil(max |d|);
 * scratch_bytes = device memory the plan holds; kernel = the a4 kernel in use (enum fdd_kernel,
 * never AUTO). */
int fdd_plan_get_info(const fdd_plan *plan, long long *nfft, long long *nbins,
                      long long *valid_len, double *max_delay_samples, size_t *scratch_bytes,
                      int *kernel);

/* Copy the plan's delay table to delay_samples_host[ndm][nchans] (HOST). */
int fdd_plan_get_delays(const fdd_plan *plan, double *delay_samples_host);

/* The time-domain comparator (the paper's "TDD"; Eq. 2) for the same
 * plan, on the same GPU: out[j][n] = sum_c in[(n + s[j][c]) mod nsamps][c], with the plan's delays
 * rounded to the nearest sample, s = floor(d + 1/2).  Exact integer sums, written as float32.
 *   in_u8  DEVICE, uint8 [nsamps][nchans] as for fdd_execute
 *   out    DEVICE, float [ndm][nsamps]; the first valid_len samples of a row are free of wrap-around
 * Asynchronous on cuda_stream.  Ignores fdd_plan_set_kernel / fdd_plan_set_decimation.  It exists
 * to put the paper's comparison (FDD against optimised time-domain dedispersion) on one machine;
 * it is not a step of the FDD path. */
int fdd_tdd_execute(fdd_plan *plan, const unsigned char *in_u8, float *out, void *cuda_stream);

/* Stage timing.  fdd_plan_set_profiling(plan, 1) makes every following execute record CUDA
 * events between the stages on its stream, and zeroes the totals; fdd_plan_get_stage_ms waits
 * for the last execute and writes the device time of each stage, summed over all executes since
 * that call, in milliseconds to ms_host[FDD_NUM_STAGES] (0 for a skipped stage) and, if
 * launches_host != NULL, how many kernels / library calls each stage launched in total (counted
 * with profiling on or off). */
int fdd_plan_set_profiling(fdd_plan *plan, int enable);
int fdd_plan_get_stage_ms(fdd_plan *plan, float *ms_host, int *launches_host);

/* Debug/test access: DEVICE pointer to the channel spectra X (float2 [nchans][pitch]) left by
 * the last execute, and the row pitch in float2 elements.  The unpack step subtracts 128 from every
 * sample (exact) so that the mean of unsigned-byte data stays out of the fp32 FFTs; *dc_removed (may
 * be NULL) receives what has to be added to Re X[c][0] of every channel to get the plain DFT
 * (128 * nsamps).  When nsamps is a power of two that is all: the sum kernel restores it in bin 0.
 * When the series is zero padded the removed mean is a rectangle, not a constant: its spectrum
 * 128 R[k], R[k] = sum_{n < nsamps} e^{-2 pi i k n / nfft}, is missing from bins k < exact_bins of X
 * (fdd_plan_get_padding; 4096, or all bins of a shorter spectrum) and already added back (closed form,
 * fp64) in the bins above; the lowest bins' share of every trial DM is tabulated per plan in fp64 and
 * added after step a4 (fdd_plan_prepare builds the table, else the first execute).  Results are those
 * of the zero-padded series (reading S9); only the fp32 rounding differs. */
int fdd_plan_get_spectrum(const fdd_plan *plan, void **x_dev, long long *pitch_elems,
                          double *dc_removed);

/* *exact_bins = number of lowest bins whose rectangle term is handled by the per-plan table (0 when
 * nsamps is a power of two). */
int fdd_plan_get_padding(const fdd_plan *plan, long long *exact_bins);

/* Run only a4 on the spectra left by the last execute (for timing sweeps of the hot kernel). */
int fdd_rotate_sum_only(fdd_plan *plan, void *out, int mode, void *cuda_stream);

/* Measure this device's FP32 FMA rate with a register-resident FFMA loop on every SM (the
 * denominator of the a4 roofline).  packed != 0 uses fma.rn.f32x2.  Writes
 * TFLOP/s (2 flop per FMA lane) and the kernel time.  Synchronous. */
int fdd_measure_fp32_peak(int packed, int iters, double *tflops_host, float *ms_host);

/* Self-test of the tensor-core path's conventions: d_dev[128][64] (float, DEVICE) = A * B^T for
 * a_f16_dev[128][64] and b_f16_dev[64][64] (IEEE half, row-major, DEVICE), through the shared-memory
 * operand layout, descriptors, tcgen05.mma sequence and TMEM read-out FDD_KERNEL_TENSOR uses. */
int fdd_tc_selftest(const void *a_f16_dev, const void *b_f16_dev, float *d_dev, void *cuda_stream);

/* Step a4 WITHOUT any allocation, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it):
 *   out[j][k] = sum_c X[c][k] exp(+2 pi i k d[j][c] / nfft)  (+ dc_add on Re out[j][0])
 * (Eq. 4 + Eq. 7; the sum FDD_MODE_FOURIER returns, any delay table).  No plan:
 *   x_dev       DEVICE, complex64 [nchans][xpitch], bins 0 .. nbins-1 of every channel's spectrum
 *               (xpitch >= nbins, in complex elements), e.g. what fdd_plan_get_spectrum returns
 *   delays_dev  DEVICE, fp64 [ndm][nchans], delays in samples (any sign, fractional)
 *   nfft        length of the transform the spectra come from (a power of two gives exact phases);
 *               nbins <= nfft / 2 + 1
 *   out_dev     DEVICE, complex64 [ndm][nbins], overwritten
 *   dc_add      added to the real part of bin 0 of every trial DM (the mean step a2 removed, or 0)
 * Caller owns every buffer; the call is asynchronous on cuda_stream (two kernels) and runs on the
 * CURRENT device, which must own the buffers.  Its only scratch - the 64-bit phase steps
 * frac(d / nfft) 2^64, [nchans][ndm rounded up to 8] - is a static __device__ array of
 * FDD_STATIC_MAX_PHASES entries (8 MiB, held by every GPU that loads the library until the process
 * exits); the call calls no cudaMalloc / cudaFree / allocating library routine (its first call on a
 * device looks the array's address up, once).  Limits and errors: FDD_ERR_TOO_LARGE if
 * nchans * round_up(ndm, 8) > FDD_STATIC_MAX_PHASES (e.g. 1024 channels x 1024 trial DMs fit) or the
 * grid would exceed 2^31 - 1 CTAs; FDD_ERR_INVALID_ARG for NULL pointers or non-positive sizes;
 * FDD_ERR_CUDA.  The array is shared by every call on a device and rewritten by each: calls that
 * overlap on the GPU (different streams or host threads) RACE - serialise them.  Speed: that of
 * FDD_KERNEL_GENERIC (one fresh phasor per element); plans remain the fast path. */
#define FDD_STATIC_MAX_PHASES 1048576
int fdd_rotate_sum_static(const void *x_dev, long long xpitch, const double *delays_dev, int nchans,
                          long long nbins, long long nfft, int ndm, void *out_dev, float dc_add,
                          void *cuda_stream);

const char *fdd_error_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* FDD_H_ */
