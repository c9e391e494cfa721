// Step a4, symmetric kernel: the fast path for DM lists that are arithmetic progressions
// within every tile of kSymT consecutive trial DMs (all five BASELINE.json configs are).
//
//   Y[j][k] = sum_c X[c][k] * exp(+2 pi i k d[j][c] / nfft)             (Eq. 4 + Eq. 7,
//                                                                   PAPER.md:64, 82)
//
// Idea.  Inside a tile the delay of row i (i = 0..T-1) on channel c is
//        d = D_c + (2 i - (T-1)) h_c            (D_c tile centre, h_c half the DM step)
// so rows come in pairs  i = T/2 + m  and  i = T/2 - 1 - m  with phasors
//        exp(i theta_c) * exp(+-i (2m+1) phi_c),   theta = 2 pi k D_c / nfft, phi = 2 pi k h_c / nfft.
// With Z = X * exp(i theta)  and  (a_m, b_m) = (cos, sin)((2m+1) phi):
//        Y+ = sum_c Z (a + i b) = (S_r + D_r) + i (S_i + D_i)
//        Y- = sum_c Z (a - i b) = (S_r - D_r) + i (S_i - D_i)
//        S_r += Z_r a   D_i += Z_r b   S_i += Z_i a   D_r += -Z_i b
// i.e. FOUR multiply-adds per PAIR of outputs instead of four per output, and the phasors follow
// from the three-term recurrence  E_{m+1} = 2 cos(2 phi) E_m - E_{m-1}  (E = (a, b)), ONE packed
// FMA per pair.  Everything is issued as packed fma.rn.f32x2 (SASS FFMA2), lanes = (a, b):
//        U_m = (S_r, D_i) += (Z_r,  Z_r) * E_m
//        V_m = (S_i, D_r) += (Z_i, -Z_i) * E_m
//        E_{m+1}          = (c2, c2) * E_m - E_{m-1}
// 3 FFMA2 = 6 FP32 lane-operations per pair = 3 per (dm, channel, bin) element, against the 8
// of a rotate-then-MAC kernel.  FFMA2 reaches the same lane throughput as scalar FFMA on B200
// with half the issue slots (measured), which leaves room for the per-(channel, bin)
// set-up below to run on the ALU / XU pipes in the shadow of the FMA pipe.
//
// Precision.  theta and phi are exact: the plan stores frac(D_c/nfft) and frac(h_c/nfft) as
// 64-bit binary fractions of a cycle (host, long double); k * P mod 2^64 is the exact fractional
// cycle, whose top 32 bits go to the SFU sine/cosine (abs. error <= 2^-21.4, no range reduction
// needed in [-pi, pi)).  c2 = 2 cos(2 phi) is formed from whichever of a_0, b_0 is smaller in
// magnitude (2 - 4 b_0^2 or 4 a_0^2 - 2), which keeps the recurrence's error bounded by about
// 3 (2m+1) * 4e-7 <= 2e-5 at the outermost pair (m = 15) and ~4e-6 rms.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>

#include <vector>

namespace fdd {

constexpr int kSymT = 32;              // trial DMs per tile
constexpr int kSymPairs = kSymT / 2;
constexpr int kSymThreads = 256;

struct SymTables {
    unsigned long long* centre64 = nullptr;   // [ntiles][nchans] frac(D_c / nfft) * 2^64
    unsigned long long* half64 = nullptr;     // [ntiles][nchans] frac(h_c / nfft) * 2^64
    int ntiles = 0;
    size_t bytes = 0;
    bool pair_ok = false;   // every adjacent pair of sub-tiles continues one progression
    // cont[t] != 0: sub-tile t + 1 continues the progression of sub-tile t (same half step, centre
    // 64 half steps on), so the two may share a CTA of fdd_kernels_sym2.cuh; host side only
    std::vector<unsigned char> cont;
    // ap[t] != 0: sub-tile t is an arithmetic progression in every channel (host side only); a DM
    // plan whose step changes inside a tile has a few tiles that are not, and those rows go to the
    // generic kernel (FDD_KERNEL_MIXED)
    std::vector<unsigned char> ap;
    int nap = 0;            // number of such tiles
};

// For every adjacent pair of sub-tiles t, t+1: do they continue one arithmetic progression in every
// channel (same half step, centre(t+1) = centre(t) + 64 half steps)?  (host, plan time)
inline void sym_continuations(const std::vector<unsigned long long>& centre64,
                              const std::vector<unsigned long long>& half64, int ntiles, int nchans,
                              std::vector<unsigned char>* cont)
{
    // units of 2^-64 cycle per bin; bins < 2^31: 2^20 is < 1e-4 cycles of phase anywhere
    auto near0 = [](unsigned long long d) { return d <= (1ULL << 20) || d >= ~0ULL - (1ULL << 20); };
    cont->assign(ntiles > 0 ? ntiles : 0, 0);
    for (int t = 0; t + 1 < ntiles; ++t) {
        bool ok = true;
        for (int c = 0; c < nchans && ok; ++c) {
            const unsigned long long ha = half64[(size_t)t * nchans + c];
            const unsigned long long hb = half64[(size_t)(t + 1) * nchans + c];
            const unsigned long long ca = centre64[(size_t)t * nchans + c];
            const unsigned long long cb = centre64[(size_t)(t + 1) * nchans + c];
            ok = near0(ha - hb) && near0(cb - ca - (ha << 6));
        }
        (*cont)[t] = ok ? 1 : 0;
    }
}

inline void sym_free_tables(SymTables* t)
{
    cudaFree(t->centre64);
    cudaFree(t->half64);
    t->centre64 = t->half64 = nullptr;
    t->ntiles = 0;
    t->bytes = 0;
    t->pair_ok = false;
    t->cont.clear();
    t->ap.clear();
    t->nap = 0;
}

inline unsigned long long sym_fixed64(long double cyc)
{
    long double f = cyc - floorl(cyc);
    long double s = f * 18446744073709551616.0L;
    if (s >= 18446744073709551615.0L) return 0ULL;
    return (unsigned long long)(s + 0.5L);
}

// Build the per-tile tables; *ok = every tile is an arithmetic progression in every channel
// (t->ap says which are; the table entries of the others are not used).  delays: host
// [ndm][nchans] in samples.
inline int sym_build_tables(SymTables* t, const double* delays, int ndm, int nchans, long long nfft,
                            bool* ok, size_t* scratch_bytes)
{
    if (scratch_bytes) *scratch_bytes -= t->bytes;
    sym_free_tables(t);
    *ok = false;
    const int ntiles = (ndm + kSymT - 1) / kSymT;
    std::vector<unsigned long long> hc((size_t)ntiles * nchans), hh((size_t)ntiles * nchans);
    t->ap.assign(ntiles, 1);
    for (int tl = 0; tl < ntiles; ++tl) {
        const int j0 = tl * kSymT;
        const int r = ndm - j0 < kSymT ? ndm - j0 : kSymT;
        for (int c = 0; c < nchans; ++c) {
            const long double d0 = delays[(size_t)j0 * nchans + c];
            // a one-row tail tile continues the step of the row before it (any step fits one row)
            const long double step =
                r >= 2 ? ((long double)delays[(size_t)(j0 + r - 1) * nchans + c] - d0) / (r - 1)
                       : (j0 > 0 ? d0 - (long double)delays[(size_t)(j0 - 1) * nchans + c] : 0.0L);
            for (int i = 1; i < r; ++i) {
                const long double want = d0 + step * i;
                const long double got = delays[(size_t)(j0 + i) * nchans + c];
                // 1e-8 samples is < 5e-9 cycles of phase at any bin
                if (fabsl(got - want) > 1e-8L) t->ap[tl] = 0;
            }
            const long double h = step / 2;
            const long double dc = d0 + (kSymT - 1) * h;
            hc[(size_t)tl * nchans + c] = sym_fixed64(dc / (long double)nfft);
            hh[(size_t)tl * nchans + c] = sym_fixed64(h / (long double)nfft);
        }
    }
    const size_t bytes = hc.size() * sizeof(unsigned long long);
    if (cudaMalloc(&t->centre64, bytes) != cudaSuccess || cudaMalloc(&t->half64, bytes) != cudaSuccess) {
        cudaGetLastError();
        sym_free_tables(t);
        return -2;
    }
    if (cudaMemcpy(t->centre64, hc.data(), bytes, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(t->half64, hh.data(), bytes, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        sym_free_tables(t);
        return -3;
    }
    t->ntiles = ntiles;
    sym_continuations(hc, hh, ntiles, nchans, &t->cont);
    t->nap = 0;
    for (int tl = 0; tl < ntiles; ++tl) {
        t->nap += t->ap[tl];
        if (!t->ap[tl]) {                              // never grouped with a neighbour
            t->cont[tl] = 0;
            if (tl > 0) t->cont[tl - 1] = 0;
        }
    }
    t->pair_ok = true;
    for (int tl = 0; tl + 1 < ntiles; ++tl) t->pair_ok = t->pair_ok && t->cont[tl];
    t->bytes = 2 * bytes;
    if (scratch_bytes) *scratch_bytes += t->bytes;
    *ok = t->nap == ntiles;
    return 0;
}

// Fractional cycle of k * P / 2^64 in [-1/2, 1/2) as radians.
__device__ __forceinline__ float sym_phase_rad(unsigned long long p64, unsigned int k)
{
    const unsigned long long t = p64 * (unsigned long long)k;        // mod 2^64: exact reduction
    return (float)(int)(unsigned int)(t >> 32) * 1.4629180792671596e-09f;   // 2 pi * 2^-32
}

struct SymSeed {
    float2 zr;      // ( Z_r,  Z_r)
    float2 zi;      // ( Z_i, -Z_i)
    float2 e0;      // (a_0, b_0)
    float2 c2;      // (c2, c2)
};

__device__ __forceinline__ SymSeed sym_seed(float2 x, unsigned long long pc, unsigned long long ph,
                                            unsigned int k)
{
    float bs, bc, b0, a0;
    __sincosf(sym_phase_rad(pc, k), &bs, &bc);
    __sincosf(sym_phase_rad(ph, k), &b0, &a0);
    const float zr = fmaf(x.x, bc, -x.y * bs);
    const float zi = fmaf(x.x, bs, x.y * bc);
    // c2 = 2 cos(2 phi) from the smaller of |a_0|, |b_0|: 2 - 4 b^2 = 4 a^2 - 2
    const float tmin = fminf(fabsf(a0), fabsf(b0));
    const float q = fmaf(-4.f * tmin, tmin, 2.f);
    const float c2 = fabsf(b0) < fabsf(a0) ? q : -q;
    SymSeed s;
    s.zr = make_float2(zr, zr);
    s.zi = make_float2(zi, -zi);
    s.e0 = make_float2(a0, b0);
    s.c2 = make_float2(c2, c2);
    return s;
}

template <int KT>
__global__ void __launch_bounds__(kSymThreads, 1)
k_rotate_sum_sym(const float2* __restrict__ X, long long xpitch,
                 const unsigned long long* __restrict__ centre64,
                 const unsigned long long* __restrict__ half64, int nchans, long long nbins,
                 int tile0, int ntiles, int ndm, float2* __restrict__ out, long long opitch,
                 int row0, float scale, int real_edges, float dc_add)
{
    // 1-D grid, DM tile fastest: CTAs resident together read the same X slab through L2.
    const int tile = tile0 + (int)(blockIdx.x % (unsigned)ntiles);
    const long long kb = blockIdx.x / (unsigned)ntiles;
    const long long kbase = kb * (kSymThreads * KT) + threadIdx.x;
    if (kbase >= nbins) return;                       // no block-wide barriers below

    long long kk[KT];
    bool live[KT];
#pragma unroll
    for (int b = 0; b < KT; ++b) {
        const long long k = kbase + (long long)b * kSymThreads;
        live[b] = k < nbins;
        kk[b] = live[b] ? k : kbase;                  // dead lanes redo bin kbase, never stored
    }

    float2 U[KT][kSymPairs], V[KT][kSymPairs];
#pragma unroll
    for (int b = 0; b < KT; ++b)
#pragma unroll
        for (int m = 0; m < kSymPairs; ++m) U[b][m] = V[b][m] = make_float2(0.f, 0.f);

    const unsigned long long* pc = centre64 + (size_t)tile * nchans;
    const unsigned long long* ph = half64 + (size_t)tile * nchans;

    // software pipeline: the seeds of channel c+1 are prepared while channel c accumulates
    SymSeed cur[KT];
#pragma unroll
    for (int b = 0; b < KT; ++b)
        cur[b] = sym_seed(X[kk[b]], __ldg(pc), __ldg(ph), (unsigned int)kk[b]);

    for (int c = 0; c < nchans; ++c) {
        const int cn = c + 1 < nchans ? c + 1 : c;
        const unsigned long long pcn = __ldg(pc + cn), phn = __ldg(ph + cn);
        float2 xn[KT];
#pragma unroll
        for (int b = 0; b < KT; ++b) xn[b] = X[(long long)cn * xpitch + kk[b]];

#pragma unroll
        for (int b = 0; b < KT; ++b) {
            float2 e = cur[b].e0;
            float2 ep = make_float2(e.x, -e.y);       // E_{-1} = conj(E_0)
#pragma unroll
            for (int m = 0; m < kSymPairs; ++m) {
                U[b][m] = __ffma2_rn(cur[b].zr, e, U[b][m]);
                V[b][m] = __ffma2_rn(cur[b].zi, e, V[b][m]);
                if (m + 1 < kSymPairs) {
                    const float2 en = __ffma2_rn(cur[b].c2, e, make_float2(-ep.x, -ep.y));
                    ep = e;
                    e = en;
                }
            }
        }
#pragma unroll
        for (int b = 0; b < KT; ++b) cur[b] = sym_seed(xn[b], pcn, phn, (unsigned int)kk[b]);
    }

    // U = (S_r, D_i), V = (S_i, D_r):  Y+ = (S_r + D_r, S_i + D_i), Y- = (S_r - D_r, S_i - D_i)
    const int j0 = tile * kSymT;
#pragma unroll
    for (int b = 0; b < KT; ++b) {
        if (!live[b]) continue;
        const long long k = kk[b];
        const bool edge = real_edges && (k == 0 || k == nbins - 1);
        const float dc = k == 0 ? dc_add : 0.f;       // the mean a2 removed (already scaled)
#pragma unroll
        for (int m = 0; m < kSymPairs; ++m) {
            const int jp = j0 + kSymPairs + m, jm = j0 + kSymPairs - 1 - m;
            if (jp < ndm)
                out[(long long)(jp - row0) * opitch + k] =
                    make_float2((U[b][m].x + V[b][m].y) * scale + dc,
                                edge ? 0.f : (V[b][m].x + U[b][m].y) * scale);
            if (jm < ndm)
                out[(long long)(jm - row0) * opitch + k] =
                    make_float2((U[b][m].x - V[b][m].y) * scale + dc,
                                edge ? 0.f : (V[b][m].x - U[b][m].y) * scale);
        }
    }
}

constexpr int kSymKT = 2;   // bins per thread

// Rows [j_begin, j_begin + rows) -> dst[(j - j_begin) * opitch + k].  j_begin must be a multiple
// of kSymT (the plan's DM chunks are).
inline int sym_launch(const SymTables& t, const float2* X, long long xpitch, int nchans,
                      long long nbins, int ndm, int j_begin, int rows, float2* dst, long long opitch,
                      float scale, int real_edges, float dc_add, cudaStream_t s)
{
    if (j_begin % kSymT != 0 || !t.centre64) return -5;
    const int tile0 = j_begin / kSymT;
    const int ntl = (rows + kSymT - 1) / kSymT;
    const int row_end = j_begin + rows < ndm ? j_begin + rows : ndm;
    const long long per_cta = (long long)kSymThreads * kSymKT;
    const long long nkb = (nbins + per_cta - 1) / per_cta;
    if ((long long)ntl * nkb > 2147483647LL) return -5;
    k_rotate_sum_sym<kSymKT><<<(unsigned)(ntl * nkb), kSymThreads, 0, s>>>(
        X, xpitch, t.centre64, t.half64, nchans, nbins, tile0, ntl, row_end, dst, opitch, j_begin,
        scale, real_edges, dc_add);
    return cudaGetLastError() == cudaSuccess ? 0 : -3;
}

}  // namespace fdd
