// Step a4, symmetric kernel with a SHARED recurrence: one CTA tile = two adjacent 32-DM
// sub-tiles (64 trial DMs) of fdd_kernels_sym.cuh's pairing.
//
//   Y[j][k] = sum_c X[c][k] * exp(+2 pi i k d[j][c] / nfft)             (Eq. 4 + Eq. 7,
//                                                                   PAPER.md:64, 82)
//
// When the half DM step h_c is the same in both sub-tiles (a uniform DM grid), the pair phasors
// E_m = (cos, sin)((2m+1) phi), phi = 2 pi k h_c / nfft, are the SAME for both; only the centre
// rotation differs:  Z_A = X e^{i theta_A},  Z_B = X e^{i theta_B}.  Per (channel, bin) the kernel
// then issues 64 accumulate FFMA2 (4 per pair, 16 pairs, 2 sub-tiles) but only 15 recurrence
// FFMA2: 79 packed FMAs per 64 trial DMs (2.47 lane-operations per (dm, channel, bin) element)
// against 94 for two independent 32-DM tiles, and the recurrence is no longer than before
// (m <= 15), so the error bound of fdd_kernels_sym.cuh is unchanged.
//
// Accumulators (U, V as in fdd_kernels_sym.cuh, but with D_r' = -D_r so that both operands are
// plain broadcasts and no negated copy of Z_i is needed):
//        U_m = (S_r, D_i ) += (Z_r, Z_r) * E_m
//        V_m = (S_i, D_r') += (Z_i, Z_i) * E_m
//        Y+ = (S_r - D_r', S_i + D_i)      Y- = (S_r + D_r', S_i - D_i)
#pragma once
#include "fdd_kernels_sym.cuh"

namespace fdd {

constexpr int kSym2Threads = 128;
constexpr int kSym2Chunk = 1024;       // channels whose phase steps are staged in shared memory

struct Sym2Seed {
    float zrA, ziA, zrB, ziB;
    float2 e0;
    float c2;
};

// Top 32 bits of (p64 * k mod 2^64) and the full product: the exact fractional cycle of k*P.
__device__ __forceinline__ unsigned long long sym2_mul(uint2 p, unsigned int k)
{
    const unsigned long long w = (unsigned long long)p.x * k;           // lo * k
    const unsigned int top = p.y * k + (unsigned int)(w >> 32);          // (hi * k + carry) mod 2^32
    return ((unsigned long long)top << 32) | (unsigned int)w;
}

__device__ __forceinline__ float sym2_rad(unsigned int top)
{
    return (float)(int)top * 1.4629180792671596e-09f;                    // 2 pi * 2^-32
}

// Seed of one (channel, bin): centre phases of sub-tiles A and B = A + 64 half steps, pair phasor
// E_0 = (cos, sin) phi and c2 = 2 cos 2 phi.
__device__ __forceinline__ Sym2Seed sym2_seed(float2 x, uint2 pa, uint2 ph, unsigned int k)
{
    const unsigned long long ta = sym2_mul(pa, k), th = sym2_mul(ph, k);
    const unsigned long long tb = ta + (th << 6);
    float sa, ca, sb, cb, b0, a0;
    __sincosf(sym2_rad((unsigned int)(ta >> 32)), &sa, &ca);
    __sincosf(sym2_rad((unsigned int)(tb >> 32)), &sb, &cb);
    __sincosf(sym2_rad((unsigned int)(th >> 32)), &b0, &a0);
    Sym2Seed s;
    s.zrA = fmaf(x.x, ca, -x.y * sa);
    s.ziA = fmaf(x.x, sa, x.y * ca);
    s.zrB = fmaf(x.x, cb, -x.y * sb);
    s.ziB = fmaf(x.x, sb, x.y * cb);
    const float tmin = fminf(fabsf(a0), fabsf(b0));
    const float q = fmaf(-4.f * tmin, tmin, 2.f);
    s.c2 = fabsf(b0) < fabsf(a0) ? q : -q;
    s.e0 = make_float2(a0, b0);
    return s;
}

__global__ void __launch_bounds__(kSym2Threads, 3)
k_rotate_sum_sym2(const float2* __restrict__ X, long long xpitch,
                  const unsigned long long* __restrict__ centre64,
                  const unsigned long long* __restrict__ half64, int nchans, long long nbins,
                  int tile0, int npairs, int ntiles_total, int ndm, float2* __restrict__ out,
                  long long opitch, int row0, float scale, int real_edges, float dc_add)
{
    // Phase steps of the channels in flight.  They are the same for every thread, so they are
    // staged once per CTA: a global load of them inside the channel loop would share a
    // scoreboard with the X prefetch and expose its full L2/HBM latency every iteration.
    __shared__ uint2 s_pa[kSym2Chunk + 1], s_ph[kSym2Chunk + 1];

    // 1-D grid, DM tile-pair fastest: CTAs resident together read the same X slab through L2.
    const int pr = (int)(blockIdx.x % (unsigned)npairs);
    const long long kb = blockIdx.x / (unsigned)npairs;
    const long long kraw = kb * kSym2Threads + threadIdx.x;
    const bool live = kraw < nbins;
    const long long k = live ? kraw : nbins - 1;      // dead lanes redo the last bin, never stored
    const int tA = tile0 + 2 * pr;
    const bool has_b = tA + 1 < ntiles_total;         // odd tail: sub-tile B is computed, not stored

    float2 UA[kSymPairs], VA[kSymPairs], UB[kSymPairs], VB[kSymPairs];
#pragma unroll
    for (int m = 0; m < kSymPairs; ++m)
        UA[m] = VA[m] = UB[m] = VB[m] = make_float2(0.f, 0.f);

    const uint2* ga = reinterpret_cast<const uint2*>(centre64 + (size_t)tA * nchans);
    const uint2* gh = reinterpret_cast<const uint2*>(half64 + (size_t)tA * nchans);
    const unsigned int ku = (unsigned int)k;
    const float2* xq = X + k + 2 * xpitch;            // channel c + 2 of the current iteration

    Sym2Seed cur;
    float2 x1;
    for (int c0 = 0; c0 < nchans; c0 += kSym2Chunk) {
        const int n = nchans - c0 < kSym2Chunk ? nchans - c0 : kSym2Chunk;
        __syncthreads();
        for (int i = threadIdx.x; i <= n; i += kSym2Threads) {
            const int cc = c0 + i < nchans ? c0 + i : nchans - 1;
            s_pa[i] = __ldg(ga + cc);
            s_ph[i] = __ldg(gh + cc);
        }
        __syncthreads();
        if (c0 == 0) {
            cur = sym2_seed(X[k], s_pa[0], s_ph[0], ku);
            x1 = X[(nchans > 1 ? xpitch : 0) + k];
        }
        for (int i = 0; i < n; ++i) {
            float2 x2 = x1;
            if (c0 + i + 2 < nchans) x2 = *xq;        // two channels ahead
            xq += xpitch;

            const float2 zrA = make_float2(cur.zrA, cur.zrA), ziA = make_float2(cur.ziA, cur.ziA);
            const float2 zrB = make_float2(cur.zrB, cur.zrB), ziB = make_float2(cur.ziB, cur.ziB);
            const float2 c2 = make_float2(cur.c2, cur.c2);
            float2 e = cur.e0;
            float2 ep = make_float2(e.x, -e.y);       // E_{-1} = conj(E_0)
#pragma unroll
            for (int m = 0; m < kSymPairs; ++m) {
                UA[m] = __ffma2_rn(zrA, e, UA[m]);
                VA[m] = __ffma2_rn(ziA, e, VA[m]);
                UB[m] = __ffma2_rn(zrB, e, UB[m]);
                VB[m] = __ffma2_rn(ziB, e, VB[m]);
                if (m + 1 < kSymPairs) {
                    const float2 en = __ffma2_rn(c2, e, make_float2(-ep.x, -ep.y));
                    ep = e;
                    e = en;
                }
            }
            cur = sym2_seed(x1, s_pa[i + 1], s_ph[i + 1], ku);
            x1 = x2;
        }
    }
    if (!live) return;

    const bool edge = real_edges && (k == 0 || k == nbins - 1);
    const float dc = k == 0 ? dc_add : 0.f;           // the mean a2 removed (already scaled)
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        if (s == 1 && !has_b) break;
        const int j0 = (tA + s) * kSymT;
#pragma unroll
        for (int m = 0; m < kSymPairs; ++m) {
            const float2 u = s ? UB[m] : UA[m], v = s ? VB[m] : VA[m];
            const int jp = j0 + kSymPairs + m, jm = j0 + kSymPairs - 1 - m;
            if (jp < ndm)
                out[(long long)(jp - row0) * opitch + k] =
                    make_float2((u.x - v.y) * scale + dc, edge ? 0.f : (v.x + u.y) * scale);
            if (jm < ndm)
                out[(long long)(jm - row0) * opitch + k] =
                    make_float2((u.x + v.y) * scale + dc, edge ? 0.f : (v.x - u.y) * scale);
        }
    }
}

// Rows [j_begin, j_begin + rows) -> dst[(j - j_begin) * opitch + k]; j_begin a multiple of 2*kSymT.
inline int sym2_launch(const SymTables& t, const float2* X, long long xpitch, int nchans,
                       long long nbins, int ndm, int j_begin, int rows, float2* dst,
                       long long opitch, float scale, int real_edges, float dc_add, cudaStream_t s)
{
    if (j_begin % (2 * kSymT) != 0 || !t.centre64) return -5;
    const int tile0 = j_begin / kSymT;
    const int ntl = (rows + kSymT - 1) / kSymT;
    const int npairs = (ntl + 1) / 2;
    const int row_end = j_begin + rows < ndm ? j_begin + rows : ndm;
    const int ntiles_total = tile0 + ntl;             // sub-tiles past this chunk are not touched
    const long long nkb = (nbins + kSym2Threads - 1) / kSym2Threads;
    if ((long long)npairs * nkb > 2147483647LL) return -5;
    k_rotate_sum_sym2<<<(unsigned)(npairs * nkb), kSym2Threads, 0, s>>>(
        X, xpitch, t.centre64, t.half64, nchans, nbins, tile0, npairs, ntiles_total, row_end, dst,
        opitch, j_begin, scale, real_edges, dc_add);
    return cudaGetLastError() == cudaSuccess ? 0 : -3;
}

}  // namespace fdd
