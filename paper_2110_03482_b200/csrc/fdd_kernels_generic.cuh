// Step a4, generic kernel: works for ANY delay table.
//
//   Y[j][k] = sum_c X[c][k] * exp(+2 pi i * frac(k * d[j][c] / nfft))      (Eq. 4 + Eq. 7,
//                                                                   PAPER.md:64, 82)
//
// Phase: the plan stores P[c][j] = round(frac(d[j][c] / nfft) * 2^64) (built on the host in
// long double).  k * P mod 2^64 is then the fractional cycle of k*d/nfft, exactly range
// reduced by integer wrap-around, with error <= k * 2^-65 cycles.  The top 32 bits, as a signed
// integer times 2^-32, are the phase in [-1/2, 1/2) cycles, which goes to the SFU sine/cosine
// (abs. error ~4e-7, no range reduction needed).  One fresh phasor per (dm, channel, bin): the
// kernel is bound by the SFU (2 MUFU per element), which is why the plan prefers the symmetric
// kernel whenever the DM grid allows it (fdd_kernels_sym.cuh).
//
// Mapping: a warp covers 32 consecutive bins (coalesced X loads and Y stores); a thread keeps DT
// trial DMs of one bin in registers; CTAs are rasterised DM-tile fastest so that CTAs running
// at the same time read the same X columns through L2.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fdd {

constexpr int kGenDT = 8;          // trial DMs per thread
constexpr int kGenThreads = 128;   // bins per CTA

__device__ __forceinline__ float phase_cycles_from_fixed(unsigned long long p64, unsigned int k)
{
    const unsigned long long t = p64 * (unsigned long long)k;     // mod 2^64
    return (float)(int)(unsigned int)(t >> 32) * 2.3283064365386963e-10f;   // * 2^-32
}

__global__ void __launch_bounds__(kGenThreads)
k_rotate_sum_generic(const float2* __restrict__ X, long long xpitch,
                     const unsigned long long* __restrict__ phase64, int ndm_pad, int nchans,
                     long long nbins, int ndm, int j_begin, int n_jtiles,
                     float2* __restrict__ out, long long opitch, float scale, int real_edges,
                     float dc_add)
{
    // 1-D grid, DM tile fastest: CTAs resident together share X columns through L2.
    const int jt = blockIdx.x % n_jtiles;
    const long long kt = blockIdx.x / n_jtiles;
    const long long k = kt * kGenThreads + threadIdx.x;
    const int j0 = j_begin + jt * kGenDT;
    const bool live = k < nbins;
    const long long kk = live ? k : 0;
    float2 acc[kGenDT];
#pragma unroll
    for (int i = 0; i < kGenDT; ++i) acc[i] = make_float2(0.f, 0.f);

    const float two_pi = 6.283185307179586f;
    for (int c = 0; c < nchans; ++c) {
        const float2 x = X[(long long)c * xpitch + kk];
        const unsigned long long* prow = phase64 + (long long)c * ndm_pad + j0;
#pragma unroll
        for (int i = 0; i < kGenDT; ++i) {
            // (a DM tile that starts off the 8-DM grid may reach past the padded row: clamp;
            //  those trial DMs are >= ndm and never stored)
            const int ii = j0 + i < ndm_pad ? i : ndm_pad - 1 - j0;
            const float ph = phase_cycles_from_fixed(__ldg(prow + ii), (unsigned int)kk);
            float s, co;
            __sincosf(ph * two_pi, &s, &co);
            acc[i].x = fmaf(x.x, co, acc[i].x);
            acc[i].x = fmaf(-x.y, s, acc[i].x);
            acc[i].y = fmaf(x.x, s, acc[i].y);
            acc[i].y = fmaf(x.y, co, acc[i].y);
        }
    }
    if (!live) return;
    const bool edge = real_edges && (k == 0 || k == nbins - 1);
#pragma unroll
    for (int i = 0; i < kGenDT; ++i) {
        const int j = j0 + i;
        if (j >= ndm) break;
        float2 v = make_float2(acc[i].x * scale + (k == 0 ? dc_add : 0.f),
                               edge ? 0.f : acc[i].y * scale);
        out[(long long)(j - j_begin) * opitch + k] = v;
    }
}

}  // namespace fdd
