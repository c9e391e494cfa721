// Zero-padded series (nsamps < nfft): keeping the mean of the 8-bit data out of fp32.
//
// Unsigned-byte data sit on a mean of 128: a 1024-channel sum is 131 072 +- 512.  When nsamps == nfft
// that mean is one Fourier bin (k = 0) and is simply left out of the transforms.  With zero padding
// it is a rectangle 128 * rect[n] (1 for n < nsamps, 0 in the padding), whose spectrum
//
//   R[k] = sum_{n < nsamps} e^{-2 pi i k n / nfft}
//        = e^{-i pi k (nsamps - 1) / nfft} sin(pi k nsamps / nfft) / sin(pi k / nfft)
//
// decays only as nfft / (pi k): in the lowest bins it is 10^3 times the noise spectrum, so fp32 errors
// of the forward transform and of the phasors (1e-6 .. 1e-5, relative to the LARGEST term) would
// swamp the data there (measured on B200, 1024 channels x 600 000 samples: trial DM 0 at 4e-4 of the
// series' rms, 4x the bar).  Instead
//   a2   subtracts 128 from the samples (exact), so the transforms see zero-mean data;
//   bins k >= K (K = 4096): 128 R[k], by the closed form in fp64, is added to every channel's
//        spectrum before a4 - there it is no larger than the noise, the usual accuracy suffices;
//   bins k <  K: the rectangle's share of the result, 128 R[k] sum_c e^{+2 pi i k d[j][c] / nfft},
//        depends on the plan only: it is tabulated once per plan in fp64 (exact 64-bit phases) and
//        added to the sums after a4.
// Mathematically the identity; readings S9, S21 of DESIGN.md are unchanged (rows ARE zero padded).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fdd {

constexpr int kPadExactBins = 4096;

// R[k] as above; arguments of the sines reduced exactly in integers (k < 2^31, nsamps < 2^32)
__device__ __forceinline__ double2 pad_rect_spectrum(unsigned long long k, unsigned long long nsamps,
                                                     unsigned long long nfft)
{
    if (k == 0) return make_double2((double)nsamps, 0.0);
    const unsigned long long m2 = 2 * nfft;
    const double a = (double)((k * (nsamps - 1)) % m2) / (double)nfft;      // [0, 2)
    const double b = (double)((k * nsamps) % m2) / (double)nfft;
    double sa, ca;
    sincospi(a, &sa, &ca);
    const double mag = sinpi(b) / sinpi((double)k / (double)nfft);
    return make_double2(ca * mag, -sa * mag);
}

// X[c][k] += amp * R[k] for k_begin <= k < nbins, all channels
__global__ void __launch_bounds__(256)
k_pad_add_rect(float2* __restrict__ X, long long xpitch, int nchans, long long k_begin, long long nbins,
               long long nsamps, long long nfft, double amp)
{
    const long long k = k_begin + (long long)blockIdx.x * 256 + threadIdx.x;
    if (k >= nbins) return;
    const double2 r = pad_rect_spectrum((unsigned long long)k, (unsigned long long)nsamps, (unsigned long long)nfft);
    const float ar = (float)(amp * r.x), ai = (float)(amp * r.y);
    const int c0 = blockIdx.y * 32;
    for (int c = c0; c < c0 + 32 && c < nchans; ++c) {
        float2 v = X[(long long)c * xpitch + k];
        v.x += ar;
        v.y += ai;
        X[(long long)c * xpitch + k] = v;
    }
}

// tab[j][k] = amp * R[k] * sum_c exp(+2 pi i frac(k P[c][j])), k < kbins; P = 64-bit binary fractions
// of a cycle per bin, [nchans][ndm_pad] (the generic kernel's table); everything in fp64
__global__ void __launch_bounds__(128)
k_pad_build_table(const unsigned long long* __restrict__ phase64, int ndm_pad, int nchans, int ndm, int kbins,
                  long long nsamps, long long nfft, double amp, float2* __restrict__ tab)
{
    const int k = blockIdx.x * 128 + threadIdx.x;
    const int j = blockIdx.y;
    if (k >= kbins || j >= ndm) return;
    double sr = 0.0, si = 0.0;
    for (int c = 0; c < nchans; ++c) {
        const unsigned long long t = phase64[(size_t)c * ndm_pad + j] * (unsigned long long)k;   // mod 2^64: exact
        const double cyc = (double)(long long)t * 5.421010862427522e-20;                       // 2^-64, [-1/2, 1/2)
        double s, co;
        sincospi(2.0 * cyc, &s, &co);
        sr += co;
        si += s;
    }
    const double2 r = pad_rect_spectrum((unsigned long long)k, (unsigned long long)nsamps, (unsigned long long)nfft);
    tab[(size_t)j * kbins + k] = make_float2((float)(amp * (r.x * sr - r.y * si)), (float)(amp * (r.x * si + r.y * sr)));
}

// out[(j - j0) * opitch + k] += scale * tab[j][k] for j0 <= j < j0 + rows, k < kuse (rows <= 65535 per launch)
__global__ void __launch_bounds__(256)
k_pad_add_table(float2* __restrict__ out, long long opitch, const float2* __restrict__ tab, int kbins, int kuse,
                int j0, int rows, float scale, int real_edges, long long nbins)
{
    const int k = blockIdx.x * 256 + threadIdx.x;
    const int j = j0 + blockIdx.y;
    if (k >= kuse || blockIdx.y >= rows) return;
    const float2 t = tab[(size_t)j * kbins + k];
    float2 v = out[(long long)(j - j0) * opitch + k];
    v.x += scale * t.x;
    // (TIME mode: an inverse real transform takes only the real part of bins 0 and nfft / 2, reading S8)
    if (!(real_edges && (k == 0 || k == nbins - 1))) v.y += scale * t.y;
    out[(long long)(j - j0) * opitch + k] = v;
}

}  // namespace fdd
