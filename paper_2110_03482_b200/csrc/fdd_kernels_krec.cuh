// Step a4 for ANY delay table, phasors by recurrence along the Fourier bins (nfft <= 2^23).
//
//   Y[j][k] = sum_c X[c][k] * exp(+2 pi i k d[j][c] / nfft)             (Eq. 4 + Eq. 7,
//                                                                   PAPER.md:64, 82)
//
// A thread owns kRecL = 8 consecutive bins of kRecDT = 8 trial DMs.  Per (channel, trial DM) it
// seeds W = exp(2 pi i k0 P) at its first bin k0 - P = frac(d / nfft), the exact fractional cycle
// from one FP64-pipe fma as in fdd_kernels_sym2.cuh - and then walks the 8 bins with
// W <- W * S,  S = exp(2 pi i P)  (a per-(channel, DM) constant the plan tabulates in fp32):
// 4 FMA for the complex MAC + 4 for the advance per (dm, channel, bin) element, against the two
// SFU operations per element that bound fdd_kernels_generic.cuh (16 lanes / clk / SM): about 2x
// faster.  Eight steps from an exactly reduced seed keep the phase error below 1e-6 rad.
//
// This is the kernel for DM lists that are not arithmetic progressions (e.g. lists whose step
// grows smoothly with DM); progressions take the 3.5x cheaper symmetric kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fdd {

constexpr int kRecDT = 8;            // trial DMs per thread
constexpr int kRecL = 8;             // consecutive bins per thread
constexpr int kRecThreads = 128;
constexpr int kRecChunk = 64;        // channels whose table rows are staged in shared memory

// p32: [nchans][ndm_pad] doubles, frac(d / nfft) in [-1/2, 1/2) times 2^(32 - pshift);
// stepS: [nchans][ndm_pad] float2, exp(2 pi i frac(d / nfft)).  ndm_pad is a multiple of kRecDT.
__global__ void __launch_bounds__(kRecThreads, 3)
k_rotate_sum_krec(const float2* __restrict__ X, long long xpitch, const double* __restrict__ p32,
                  const float2* __restrict__ stepS, int ndm_pad, int nchans, long long nbins, int ndm,
                  int j_begin, int n_jtiles, float2* __restrict__ out, long long opitch, float scale,
                  int real_edges, float dc_add, int pshift)
{
    __shared__ double s_p[kRecChunk][kRecDT];
    __shared__ float2 s_s[kRecChunk][kRecDT];

    // 1-D grid, DM tile fastest: CTAs resident together share X columns through L2.
    const int jt = blockIdx.x % n_jtiles;
    const long long kt = blockIdx.x / n_jtiles;
    const long long k0 = (kt * kRecThreads + threadIdx.x) * kRecL;
    const int j0 = j_begin + jt * kRecDT;
    const bool live = k0 < nbins;
    const long long kk = live ? k0 : 0;
    const double kd = (double)kk;

    float2 acc[kRecDT][kRecL];
#pragma unroll
    for (int i = 0; i < kRecDT; ++i)
#pragma unroll
        for (int b = 0; b < kRecL; ++b) acc[i][b] = make_float2(0.f, 0.f);

    for (int c0 = 0; c0 < nchans; c0 += kRecChunk) {
        const int n = nchans - c0 < kRecChunk ? nchans - c0 : kRecChunk;
        __syncthreads();
        for (int i = threadIdx.x; i < n * kRecDT; i += kRecThreads) {
            const int cc = i / kRecDT, jj = i % kRecDT;
            s_p[cc][jj] = p32[(long long)(c0 + cc) * ndm_pad + j0 + jj];
            s_s[cc][jj] = stepS[(long long)(c0 + cc) * ndm_pad + j0 + jj];
        }
        __syncthreads();
        for (int cc = 0; cc < n; ++cc) {
            // the thread's 8 bins of this channel (bins past the row's pitch are never stored)
            const float2* xp = X + (long long)(c0 + cc) * xpitch + kk;
            float2 x[kRecL];
#pragma unroll
            for (int b = 0; b < kRecL; b += 2) {
                const float4 v = *reinterpret_cast<const float4*>(xp + b);
                x[b] = make_float2(v.x, v.y);
                x[b + 1] = make_float2(v.z, v.w);
            }
#pragma unroll
            for (int i = 0; i < kRecDT; ++i) {
                const unsigned int ph =
                    (unsigned int)__double2loint(fma(kd, s_p[cc][i], 6755399441055744.0)) << pshift;
                float ws, wc;
                __sincosf((float)(int)ph * 1.4629180792671596e-09f, &ws, &wc);   // 2 pi * 2^-32
                const float2 S = s_s[cc][i];
#pragma unroll
                for (int b = 0; b < kRecL; ++b) {
                    acc[i][b].x = fmaf(x[b].x, wc, acc[i][b].x);
                    acc[i][b].x = fmaf(-x[b].y, ws, acc[i][b].x);
                    acc[i][b].y = fmaf(x[b].x, ws, acc[i][b].y);
                    acc[i][b].y = fmaf(x[b].y, wc, acc[i][b].y);
                    if (b + 1 < kRecL) {
                        const float nc = fmaf(wc, S.x, -ws * S.y);
                        ws = fmaf(wc, S.y, ws * S.x);
                        wc = nc;
                    }
                }
            }
        }
    }
    if (!live) return;
#pragma unroll
    for (int i = 0; i < kRecDT; ++i) {
        const int j = j0 + i;
        if (j >= ndm) break;
#pragma unroll
        for (int b = 0; b < kRecL; ++b) {
            const long long k = k0 + b;
            if (k >= nbins) break;
            const bool edge = real_edges && (k == 0 || k == nbins - 1);
            out[(long long)(j - j_begin) * opitch + k] =
                make_float2(acc[i][b].x * scale + (k == 0 ? dc_add : 0.f), edge ? 0.f : acc[i][b].y * scale);
        }
    }
}

}  // namespace fdd
