// Row f4: the time-domain comparator ("TDD"; Eq. 2) on the same GPU.
//
//   out[j][n] = sum_c in[(n + s[j][c]) mod nsamps][c],   s = floor(d + 1/2)  (nearest sample)
//
// Two kernels, as in the paper's optimised TDD (fused unpack + transpose, then shift-and-add):
//   k_tdd_transpose  u8 [nsamps][nchans] -> u8 [nchans][tpitch]; the series is continued
//                    periodically past nsamps (tpitch >= nsamps + largest shift + 128), so the
//                    adder never wraps an index.  The data stay 8-bit: a quarter of the traffic
//                    of a float copy, and the sums are exact integers.
//   k_tdd_shift_add  CTA = 32 trial DMs (the lanes of a warp) x 256 samples (8 warps x 32).  Per
//                    channel a thread reads its 32 samples as 9 words at the byte offset of its
//                    own shift - adjacent lanes (adjacent DMs) read almost the same bytes, so the
//                    loads hit L1 - aligns them with a funnel shift and adds them four at a time
//                    into packed 16-bit lanes (2 PRMT + 2 IADD per 4 samples), spilling to 32-bit
//                    sums every 256 channels.  The words of channel c + 1 and the shift of c + 2
//                    are requested before channel c is added.  Bound by the integer ALU (1.25 operations per
//                    (dm, channel, sample)), not by HBM: the transposed input is read once through
//                    L2 per DM tile (grid is DM-tile fastest).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fdd {

constexpr int kTddDms = 32;                          // trial DMs per CTA = lanes
constexpr int kTddWarps = 8;
constexpr int kTddSeg = 32;                          // samples per thread
constexpr int kTddTile = kTddWarps * kTddSeg;        // samples per CTA
constexpr int kTddFlush = 256;                       // channels per 16-bit accumulation run

// 64 x 64 byte tiles through shared memory; out[c][n] = in[n mod nsamps][c] for n < tpitch.
__global__ void __launch_bounds__(256)
k_tdd_transpose(const unsigned char* __restrict__ in, unsigned char* __restrict__ out, int nchans,
                long long nsamps, long long tpitch)
{
    __shared__ unsigned char tile[64][64 + 4];
    const long long n0 = (long long)blockIdx.x * 64;
    const int c0 = blockIdx.y * 64;
    for (int i = threadIdx.x; i < 64 * 64; i += 256) {
        const int r = i >> 6, cc = i & 63;
        const long long n = n0 + r;
        unsigned char v = 0;
        if (n < tpitch && c0 + cc < nchans) v = in[(n % nsamps) * nchans + c0 + cc];
        tile[r][cc] = v;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 64 * 16; i += 256) {
        const int cc = i >> 4, q = i & 15;               // channel, group of 4 samples
        const long long n = n0 + 4 * q;
        if (c0 + cc < nchans && n < tpitch) {            // tpitch is a multiple of 64
            const unsigned int w = tile[4 * q][cc] | (tile[4 * q + 1][cc] << 8) |
                                   (tile[4 * q + 2][cc] << 16) | ((unsigned int)tile[4 * q + 3][cc] << 24);
            *reinterpret_cast<unsigned int*>(out + (long long)(c0 + cc) * tpitch + n) = w;
        }
    }
}

// shifts_t: [nchans][ndm_pad] non-negative shifts (already reduced mod nsamps).
__global__ void __launch_bounds__(kTddWarps * 32, 3)
k_tdd_shift_add(const unsigned char* __restrict__ xt, long long tpitch,
                const int* __restrict__ shifts_t, int ndm_pad, int nchans, long long nsamps, int ndm,
                int ntiles_dm, float* __restrict__ out)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tile_dm = blockIdx.x % ntiles_dm;          // DM tile fastest: shared rows of xt in L2
    const long long tblk = blockIdx.x / ntiles_dm;
    const int j = tile_dm * kTddDms + lane;
    const long long n0 = tblk * kTddTile + (long long)warp * kTddSeg;
    if (n0 >= nsamps) return;                            // no barriers below

    int acc[kTddSeg];
    unsigned int lo[kTddSeg / 4], hi[kTddSeg / 4];
#pragma unroll
    for (int i = 0; i < kTddSeg; ++i) acc[i] = 0;
#pragma unroll
    for (int i = 0; i < kTddSeg / 4; ++i) lo[i] = hi[i] = 0;

    const int* srow = shifts_t + (j < ndm ? j : ndm - 1);
    const unsigned char* row = xt + n0;
    constexpr int NW = kTddSeg / 4 + 1;
    // software pipeline: words of channel c + 1 and the shift of channel c + 2 are in flight while
    // channel c is added
    unsigned int wn[NW];
    unsigned int shn;
    {
        const int s0 = __ldg(srow);
        const uintptr_t a = reinterpret_cast<uintptr_t>(row) + (unsigned int)s0;
        const unsigned int* wp = reinterpret_cast<const unsigned int*>(a & ~(uintptr_t)3);
        shn = ((unsigned int)a & 3u) * 8u;
#pragma unroll
        for (int i = 0; i < NW; ++i) wn[i] = __ldg(wp + i);
    }
    int s1 = nchans > 1 ? __ldg(srow + ndm_pad) : 0;     // shift of channel c + 1
    srow += 2 * (long long)ndm_pad;                      // -> channel c + 2
    int run = 0;
#pragma unroll 2
    for (int c = 0; c < nchans; ++c) {
        unsigned int w[NW];
#pragma unroll
        for (int i = 0; i < NW; ++i) w[i] = wn[i];
        const unsigned int sh = shn;
        row += tpitch;
        if (c + 1 < nchans) {
            const uintptr_t a = reinterpret_cast<uintptr_t>(row) + (unsigned int)s1;
            const unsigned int* wp = reinterpret_cast<const unsigned int*>(a & ~(uintptr_t)3);
            shn = ((unsigned int)a & 3u) * 8u;
#pragma unroll
            for (int i = 0; i < NW; ++i) wn[i] = __ldg(wp + i);
            if (c + 2 < nchans) s1 = __ldg(srow);
            srow += ndm_pad;
        }
#pragma unroll
        for (int i = 0; i < kTddSeg / 4; ++i) {
            const unsigned int v = __funnelshift_r(w[i], w[i + 1], sh);      // 4 aligned samples
            lo[i] += __byte_perm(v, 0, 0x4240);                               // (b0, b2) as 16-bit lanes
            hi[i] += __byte_perm(v, 0, 0x4341);                               // (b1, b3)
        }
        if (++run == kTddFlush || c + 1 == nchans) {                          // 256 * 255 < 2^16
#pragma unroll
            for (int i = 0; i < kTddSeg / 4; ++i) {
                acc[4 * i + 0] += lo[i] & 0xffffu;
                acc[4 * i + 1] += hi[i] & 0xffffu;
                acc[4 * i + 2] += lo[i] >> 16;
                acc[4 * i + 3] += hi[i] >> 16;
                lo[i] = hi[i] = 0;
            }
            run = 0;
        }
    }
    if (j >= ndm) return;
    float* orow = out + (long long)j * nsamps + n0;
    const bool vec = (nsamps % 4 == 0) && n0 + kTddSeg <= nsamps;
#pragma unroll
    for (int i = 0; i < kTddSeg / 4; ++i) {
        if (vec) {
            *reinterpret_cast<float4*>(orow + 4 * i) =
                make_float4((float)acc[4 * i], (float)acc[4 * i + 1], (float)acc[4 * i + 2],
                            (float)acc[4 * i + 3]);
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (n0 + 4 * i + q < nsamps) orow[4 * i + q] = (float)acc[4 * i + q];
        }
    }
}

}  // namespace fdd
