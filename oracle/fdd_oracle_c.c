/* CPU oracle, C part -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/fdd_oracle.py).
 *
 * The same step O4 as fdd_oracle.phase_rotate_sum, written as plain loops so that the
 * at-scale tier (1024 channels x 2^20 samples, a handful of DM rows) finishes in seconds:
 *
 *   Y[j][i] = sum_c X[c][i] * exp(+2 pi i * frac(k_i * d[j][c] / N))        (Eq. 4 + Eq. 7,
 *                                                          /root/reference/PAPER.md:64, 82)
 *
 * k_i = bins[i] (or i when bins == NULL).  The product k*d/N is formed in long double
 * (64-bit mantissa on x86) and reduced to [-1/2, 1/2] cycles before the cast to double, so
 * the phase is exact to ~1e-15 cycles even at 2e4 cycles (config 5).  Sign: reading S1 of
 * fdd_oracle.py (advance by the delay with a forward kernel e^{-2 pi i k n / N}).
 *
 * Shares nothing with the CUDA path.  Pinned against the numpy definition in
 * tests/test_oracle_pins.py (test_c_matches_numpy).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* X: complex128 [nchans][nb] as (re, im) pairs; delays: [nrows][nchans] samples;
 * Y: complex128 [nrows][nb] (overwritten unless accumulate != 0). */
void oracle_phase_rotate_sum(const double *X, const double *delays, const int64_t *bins,
                             int64_t nchans, int64_t nb, int64_t nrows, int64_t nfft,
                             int accumulate, double *Y)
{
    const double two_pi = 6.283185307179586476925286766559;
    for (int64_t j = 0; j < nrows; ++j) {
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < nb; ++i) {
            const long double k = (long double)(bins ? bins[i] : i);
            double acc_re = accumulate ? Y[2 * (j * nb + i)] : 0.0;
            double acc_im = accumulate ? Y[2 * (j * nb + i) + 1] : 0.0;
            for (int64_t c = 0; c < nchans; ++c) {
                long double cyc = k * (long double)delays[j * nchans + c] / (long double)nfft;
                cyc -= rintl(cyc);
                const double ang = two_pi * (double)cyc;
                const double wr = cos(ang), wi = sin(ang);
                const double xr = X[2 * (c * nb + i)], xi = X[2 * (c * nb + i) + 1];
                acc_re += xr * wr - xi * wi;
                acc_im += xr * wi + xi * wr;
            }
            Y[2 * (j * nb + i)] = acc_re;
            Y[2 * (j * nb + i) + 1] = acc_im;
        }
    }
}
