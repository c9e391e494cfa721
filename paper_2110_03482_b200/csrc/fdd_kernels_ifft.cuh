// Step a5, hand-written: the inverse real transform of nfft points as a half-length complex transform
// in TWO passes over the data (Eq. 6), for nfft = 2^7 .. 2^23.
//
//   Z[k]  = (Y[k] + conj Y[M - k]) + i e^{+2 pi i k / N} (Y[k] - conj Y[M - k]),  k < M = N / 2
//   z[n]  = sum_k Z[k] e^{+2 pi i k n / M},     y[2n] = Re z[n],  y[2n + 1] = Im z[n]
//
// with k = M2 k1 + k2, n = n1 + M1 n2 (M = M1 M2):
//
//   pass A  B[n1][k2] = e^{+2 pi i k2 n1 / M} sum_k1 Z[M2 k1 + k2] e^{+2 pi i k1 n1 / M1}
//   pass B  z[n1 + M1 n2] = sum_k2 B[n1][k2] e^{+2 pi i k2 n2 / M2}
//
// Pass A reads Y once (its own run of C adjacent bins k2 and the mirrored run, for every k1), forms Z on
// the fly - cuFFT's C2R spends a pass of its own on that - and writes B; pass B reads B, and writes the
// real series once, adding the mean of the series that step a4 then leaves out of bin 0 (the fp32
// transform works on a series of rms sigma instead of 256 sigma).  B lives in a small ring that both
// passes go through batch by batch, so that it can stay in the 126 MB L2 and HBM sees Y once and y once.
//
// Both passes run the same transform of L = M1 or M2 points, C of them side by side in a CTA (C adjacent
// columns = one run of 8 C bytes per global row): a Stockham autosort transform whose radix-8 butterflies
// live in registers - a thread holds the 8 points t + q L / 8, q < 8, of one column; between stages the
// points are exchanged through a shared-memory tile [L][C + 1]; log2 L not a multiple of 3: one radix-2
// or radix-4 stage first (Ns = 1, no twiddles).  The first stage loads straight from global memory and
// the last one stores straight to it.  Round 2's first version kept the data in shared memory and ran
// radix-4 stages there: 56 ms at 4096 x 2^20 against cuFFT's 21 ms (instruction- and latency-bound).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

namespace fdd {

__device__ __forceinline__ float2 ifft_cmul(float2 a, float2 b)
{
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// (packed fp32 pairs: one FADD2 per complex sum)
__device__ __forceinline__ float2 ifft_add(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 ifft_sub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }

// Butterflies with the kernel e^{+2 pi i p q / R}, in place, outputs in natural order
__device__ __forceinline__ void ifft_bf2(float2& a, float2& b)
{
    const float2 t = a;
    a = ifft_add(t, b);
    b = ifft_sub(t, b);
}
__device__ __forceinline__ void ifft_bf4(float2& y0, float2& y1, float2& y2, float2& y3)
{
    const float2 s02 = ifft_add(y0, y2), d02 = ifft_sub(y0, y2);
    const float2 s13 = ifft_add(y1, y3), d13 = ifft_sub(y1, y3);
    y0 = ifft_add(s02, s13);
    y2 = ifft_sub(s02, s13);
    y1 = make_float2(d02.x - d13.y, d02.y + d13.x);      // d02 + i d13
    y3 = make_float2(d02.x + d13.y, d02.y - d13.x);      // d02 - i d13
}
__device__ __forceinline__ void ifft_bf8(float2 (&v)[8])
{
    // X[p] = A[p & 3] + w^p B[p & 3], A = DFT4(even), B = DFT4(odd), w = e^{i pi / 4}
    ifft_bf4(v[0], v[2], v[4], v[6]);                    // A0..A3 in v[0], v[2], v[4], v[6]
    ifft_bf4(v[1], v[3], v[5], v[7]);                    // B0..B3 in v[1], v[3], v[5], v[7]
    const float h = 0.70710678118654752f;
    const float2 b0 = v[1];
    const float2 b1 = make_float2((v[3].x - v[3].y) * h, (v[3].x + v[3].y) * h);     // (1 + i) / sqrt 2
    const float2 b2 = make_float2(-v[5].y, v[5].x);                                  // i
    const float2 b3 = make_float2(-(v[7].x + v[7].y) * h, (v[7].x - v[7].y) * h);    // (-1 + i) / sqrt 2
    const float2 a0 = v[0], a1 = v[2], a2 = v[4], a3 = v[6];
    v[0] = ifft_add(a0, b0); v[4] = ifft_sub(a0, b0);
    v[1] = ifft_add(a1, b1); v[5] = ifft_sub(a1, b1);
    v[2] = ifft_add(a2, b2); v[6] = ifft_sub(a2, b2);
    v[3] = ifft_add(a3, b3); v[7] = ifft_sub(a3, b3);
}

// The transform of one column: v[q] = point t + q L / 8 of the input on entry; the results are handed
// to emit(r, index, value), r = 0 .. 7 in turn.  s: tile [rows][C + 1] shared by the CTA's C columns;
// tw[j] = e^{+2 pi i j / L}.
// Stockham: a radix-R stage with Ns = product of the earlier radices takes butterfly j (< L / R) from the
// points j + r L / R, twiddles them by e^{2 pi i r k / (Ns R)}, k = j mod Ns, and puts the outputs at
// (j - k) R + k + r Ns.  Every CTA thread must call it (it synchronises the CTA).
// (t_in, c_in): the thread's role up to the first exchange, (t, c) after it - the exchange goes through
// the tile, so a thread may pick up another part of the work there (pass B loads rows along t and
// stores along c).  Tile: [L + L / 2^PAD][C], point i in row i + (i >> PAD): with the shifts ifft_pad_a / _b
// choose, a warp's 32 accesses fall on all banks evenly in (nearly) every exchange (checked by
// enumerating the access patterns: 1.0 .. 1.17 x the ideal number of wavefronts, against 1.75 .. 2 x
// for a tile with one padding column).
template <int PAD>
__device__ __forceinline__ int ifft_row(int i) { return i + (i >> PAD); }
__host__ __device__ constexpr int ifft_pad_a(int lg, int lgc) { return lgc == 3 ? (lg % 3 ? lg % 3 : 3) : 2; }
__host__ __device__ constexpr int ifft_pad_b(int lg, int lgc) { return lg >= 6 ? 3 : ifft_pad_a(lg, lgc); }

// row of point i0 + d, d a compile-time multiple: where the padding is linear in d (d a multiple of 2^PAD, or
// i0 a multiple of 2^PAD and d below it) the offset is a constant the compiler folds into the access
template <int PAD>
__device__ __forceinline__ int ifft_row_at(int row_i0, int i0, int d, bool linear)
{
    return linear ? row_i0 + d + (d >> PAD) : ifft_row<PAD>(i0 + d);
}

// ACC: every twiddle straight from a table (zero-padded series keep their mean - a rectangle 256 sigma high -
// inside the transform, and at 2^23 points the products and recurrences that save table loads cost the
// margin: max error 1.04e-3 of the rms against 0.98e-3; without padding the mean is outside, either passes
// with a wide margin and the cheaper form is 1.7 ms faster at 4096 x 2^20)
template <int LG, int LGC, int PAD, bool ACC, class Emit>
__device__ __forceinline__ void ifft_core(float2 (&v)[8], float2* s, const float2* tw, int t_in, int c_in, int t,
                                          int c, Emit emit)
{
    constexpr int L = 1 << LG, T = L / 8, P = 1 << LGC;
    constexpr int R0 = 1 << (LG % 3), N8 = LG / 3;
    bool wrote = false;
    if (R0 == 2) {
        // four radix-2 butterflies u: points v[u], v[u + 4] of butterfly j = t + u T -> 2 j, 2 j + 1
#pragma unroll
        for (int u = 0; u < 4; ++u) ifft_bf2(v[u], v[u + 4]);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            s[ifft_row<PAD>(2 * (t_in + u * T)) * P + c_in] = v[u];
            s[ifft_row<PAD>(2 * (t_in + u * T) + 1) * P + c_in] = v[u + 4];
        }
        wrote = true;
    } else if (R0 == 4) {
        // two radix-4 butterflies u: points v[u + 2 r] of butterfly j = t + u T -> 4 j + r
#pragma unroll
        for (int u = 0; u < 2; ++u) ifft_bf4(v[u], v[u + 2], v[u + 4], v[u + 6]);
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
            for (int r = 0; r < 4; ++r) s[ifft_row<PAD>(4 * (t_in + u * T) + r) * P + c_in] = v[u + 2 * r];
        wrote = true;
    }
    if (wrote) {
        __syncthreads();
        {
            const int rt = ifft_row<PAD>(t);
#pragma unroll
            for (int q = 0; q < 8; ++q) v[q] = s[ifft_row_at<PAD>(rt, t, q * T, T % (1 << PAD) == 0) * P + c];
        }
    }
#pragma unroll
    for (int i = 0; i < N8; ++i) {
        const int Ns = R0 << (3 * i);
        const int tt = wrote ? t : t_in, cc = wrote ? c : c_in;
        const int k = tt & (Ns - 1);
        if (Ns > 1) {
            // w^r, r = 1 .. 7, w = e^{2 pi i k / (8 Ns)}: three from the table, four products
            const int step = L / (8 * Ns);
            const float2 w1 = tw[k * step], w2 = tw[2 * k * step], w4 = tw[4 * k * step];
            const float2 w3 = ACC ? tw[3 * k * step] : ifft_cmul(w1, w2);
            const float2 w5 = ACC ? tw[5 * k * step] : ifft_cmul(w1, w4);
            const float2 w6 = ACC ? tw[6 * k * step] : ifft_cmul(w2, w4);
            const float2 w7 = ACC ? tw[7 * k * step] : ifft_cmul(w3, w4);
            v[1] = ifft_cmul(v[1], w1); v[2] = ifft_cmul(v[2], w2); v[3] = ifft_cmul(v[3], w3);
            v[4] = ifft_cmul(v[4], w4); v[5] = ifft_cmul(v[5], w5); v[6] = ifft_cmul(v[6], w6);
            v[7] = ifft_cmul(v[7], w7);
        }
        ifft_bf8(v);
        const int j0 = (tt - k) * 8 + k;
        if (i == N8 - 1) {
#pragma unroll
            for (int r = 0; r < 8; ++r) emit(r, j0 + r * Ns, v[r]);
        } else {
            if (wrote) __syncthreads();              // the reads of the stage before are done
            {
                // (Ns a multiple of 2^PAD: linear; Ns = 1 with 2^PAD >= 8: j0 = 8 t is a multiple of 8 and r < 8)
                const int rj = ifft_row<PAD>(j0);
                const bool lin = Ns % (1 << PAD) == 0 || (Ns == 1 && PAD >= 3);
#pragma unroll
                for (int r = 0; r < 8; ++r) s[ifft_row_at<PAD>(rj, j0, r * Ns, lin) * P + cc] = v[r];
            }
            wrote = true;
            __syncthreads();
            {
                const int rt = ifft_row<PAD>(t);
#pragma unroll
                for (int q = 0; q < 8; ++q) v[q] = s[ifft_row_at<PAD>(rt, t, q * T, T % (1 << PAD) == 0) * P + c];
            }
        }
    }
}

// Two transforms per thread (columns 2 c and 2 c + 1 of a tile [rows][2 C], moved as one 16-byte access;
// one set of twiddles for both): same stages as ifft_core, no change of roles.
template <int LG, int LGC, int PAD, bool ACC, class Emit>
__device__ __forceinline__ void ifft_core2(float2 (&va)[8], float2 (&vb)[8], float2* s, const float2* tw, int t, int c,
                                           Emit emit)
{
    constexpr int L = 1 << LG, T = L / 8, P4 = 1 << LGC;       // float4 per tile row
    constexpr int R0 = 1 << (LG % 3), N8 = LG / 3;
    float4* s4 = reinterpret_cast<float4*>(s);
    auto put = [&](int row, float2 a, float2 b) { s4[row * P4 + c] = make_float4(a.x, a.y, b.x, b.y); };
    auto get = [&](int row, float2& a, float2& b) {
        const float4 w = s4[row * P4 + c];
        a = make_float2(w.x, w.y);
        b = make_float2(w.z, w.w);
    };
    bool wrote = false;
    if (R0 == 2) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            ifft_bf2(va[u], va[u + 4]);
            ifft_bf2(vb[u], vb[u + 4]);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            put(ifft_row<PAD>(2 * (t + u * T)), va[u], vb[u]);
            put(ifft_row<PAD>(2 * (t + u * T) + 1), va[u + 4], vb[u + 4]);
        }
        wrote = true;
    } else if (R0 == 4) {
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            ifft_bf4(va[u], va[u + 2], va[u + 4], va[u + 6]);
            ifft_bf4(vb[u], vb[u + 2], vb[u + 4], vb[u + 6]);
        }
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
            for (int r = 0; r < 4; ++r) put(ifft_row<PAD>(4 * (t + u * T) + r), va[u + 2 * r], vb[u + 2 * r]);
        wrote = true;
    }
    if (wrote) {
        __syncthreads();
        const int rt = ifft_row<PAD>(t);
#pragma unroll
        for (int q = 0; q < 8; ++q) get(ifft_row_at<PAD>(rt, t, q * T, T % (1 << PAD) == 0), va[q], vb[q]);
    }
#pragma unroll
    for (int i = 0; i < N8; ++i) {
        const int Ns = R0 << (3 * i);
        const int k = t & (Ns - 1);
        if (Ns > 1) {
            const int step = L / (8 * Ns);
            const float2 w1 = tw[k * step], w2 = tw[2 * k * step], w4 = tw[4 * k * step];
            const float2 w3 = ACC ? tw[3 * k * step] : ifft_cmul(w1, w2);
            const float2 w5 = ACC ? tw[5 * k * step] : ifft_cmul(w1, w4);
            const float2 w6 = ACC ? tw[6 * k * step] : ifft_cmul(w2, w4);
            const float2 w7 = ACC ? tw[7 * k * step] : ifft_cmul(w3, w4);
            va[1] = ifft_cmul(va[1], w1); va[2] = ifft_cmul(va[2], w2); va[3] = ifft_cmul(va[3], w3);
            va[4] = ifft_cmul(va[4], w4); va[5] = ifft_cmul(va[5], w5); va[6] = ifft_cmul(va[6], w6);
            va[7] = ifft_cmul(va[7], w7);
            vb[1] = ifft_cmul(vb[1], w1); vb[2] = ifft_cmul(vb[2], w2); vb[3] = ifft_cmul(vb[3], w3);
            vb[4] = ifft_cmul(vb[4], w4); vb[5] = ifft_cmul(vb[5], w5); vb[6] = ifft_cmul(vb[6], w6);
            vb[7] = ifft_cmul(vb[7], w7);
        }
        ifft_bf8(va);
        ifft_bf8(vb);
        const int j0 = (t - k) * 8 + k;
        if (i == N8 - 1) {
#pragma unroll
            for (int r = 0; r < 8; ++r) emit(r, j0 + r * Ns, va[r], vb[r]);
        } else {
            if (wrote) __syncthreads();
            {
                const int rj = ifft_row<PAD>(j0);
                const bool lin = Ns % (1 << PAD) == 0 || (Ns == 1 && PAD >= 3);
#pragma unroll
                for (int r = 0; r < 8; ++r) put(ifft_row_at<PAD>(rj, j0, r * Ns, lin), va[r], vb[r]);
            }
            wrote = true;
            __syncthreads();
            {
                const int rt = ifft_row<PAD>(t);
#pragma unroll
                for (int q = 0; q < 8; ++q) get(ifft_row_at<PAD>(rt, t, q * T, T % (1 << PAD) == 0), va[q], vb[q]);
            }
        }
    }
}

// tw[j] = e^{+2 pi i j / L}, j < L (the quotient is exact in fp32)
__device__ __forceinline__ void ifft_make_twiddles(float2* tw, int L, int nthreads)
{
    for (int j = threadIdx.x; j < L; j += nthreads) {
        float sn, cs;
        sincospif(2.f * (float)j / (float)L, &sn, &cs);
        tw[j] = make_float2(cs, sn);
    }
}

__host__ __device__ constexpr int ifft_hi_len(int lg) { return lg > 5 ? 1 << (lg - 5) : 1; }

// shared memory of the two passes, in float2 elements
constexpr size_t ifft_smem_a(int lg, int lgc)
{
    return ((size_t)((1 << lg) + ((1 << lg) >> ifft_pad_a(lg, lgc))) * (1 << lgc) + 2 * (size_t)(1 << lg) +
            (size_t)(1 << lgc) * (ifft_hi_len(lg) + 34)) * sizeof(float2);
}
constexpr size_t ifft_smem_b(int lg, int lgc)
{
    return ((size_t)((1 << lg) + ((1 << lg) >> ifft_pad_b(lg, lgc))) * (1 << lgc) + (size_t)(1 << lg)) * sizeof(float2);
}

// Per-plan twiddle tables (a sincospif per CTA thread and table entry costs 13 % of the passes'
// instructions): [tw1: L1][half: L1][tw2: L2][per column k2 < M2: hi (HI), lo (32), colw, colg], float2.
//   tw[j]   = e^{2 pi i j / L}          half[j] = e^{i pi j / L1}
//   e^{i pi k / M},        k = M2 k1 + k2:  half[k1] times colw[k2] = e^{i pi k2 / M}
//   e^{2 pi i k2 n1 / M},  n1 = 32 a + b:   hi[k2][a] = e^{2 pi i k2 32 a / M} times lo[k2][b] = e^{2 pi i k2 b / M};
//                                           colg[k2] = e^{2 pi i k2 (L1 / 8) / M} steps n1 by L1 / 8
inline size_t ifft_table_elems(int lg1, int lg2)
{
    return 2 * ((size_t)1 << lg1) + ((size_t)1 << lg2) + ((size_t)1 << lg2) * (ifft_hi_len(lg1) + 34);
}

__global__ void __launch_bounds__(256) k_ifft_tables(float2* tab, int lg1, int lg2)
{
    const long long L1 = 1LL << lg1, L2 = 1LL << lg2, M = L1 * L2;
    const int HI = lg1 > 5 ? 1 << (lg1 - 5) : 1, W = HI + 34;
    const long long n = 2 * L1 + L2 + L2 * W;
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    double arg;                                     // in half turns (sincospi)
    if (i < L1) arg = 2.0 * (double)i / (double)L1;
    else if (i < 2 * L1) arg = (double)(i - L1) / (double)L1;
    else if (i < 2 * L1 + L2) arg = 2.0 * (double)(i - 2 * L1) / (double)L2;
    else {
        const long long e = i - 2 * L1 - L2, k2 = e / W, r = e - k2 * W;
        if (r < HI) arg = 2.0 * (double)((k2 * 32 * r) % M) / (double)M;
        else if (r < HI + 32) arg = 2.0 * (double)(k2 * (r - HI)) / (double)M;
        else if (r == HI + 32) arg = (double)k2 / (double)M;
        else arg = 2.0 * (double)((k2 * (L1 / 8)) % M) / (double)M;
    }
    double sn, cs;
    sincospi(arg, &sn, &cs);
    tab[i] = make_float2((float)cs, (float)sn);
}

// Pass A.  grid = (M2 / C, rows), CTA = C columns x L / 8 threads, L = M1 = 2^LG.
// Y: [rows][ypitch] sums of a4 (bins 0 .. M); B: [rows][M] as [n1][k2].
// Twiddles come from small per-CTA tables (a sincospif per element would cost as much as the transform):
//   e^{i pi k / M},        k = M2 k1 + k2:  half[k1] = e^{i pi k1 / M1}  times  colw[c] = e^{i pi k2 / M}
//   e^{2 pi i k2 n1 / M},  n1 = 32 a + b:   hi[c][a] = e^{2 pi i k2 32 a / M}  times  lo[c][b] = e^{2 pi i k2 b / M}
#ifndef IFFT_MINB_A
#define IFFT_MINB_A 2
#endif
#ifndef IFFT_MINB_B
#define IFFT_MINB_B 2
#endif
template <int LG, int LGC, bool ACC>
__global__ void __launch_bounds__(1 << (LG - 3 + LGC), (LG - 3 + LGC) >= 10 ? 1 : IFFT_MINB_A)
k_ifft_pass_a(const float2* __restrict__ Y, long long ypitch, float2* __restrict__ B, int lg2,
              const float2* __restrict__ tab)
{
    constexpr int L = 1 << LG, C = 1 << LGC, T = L / 8, NT = T * C, HI = ifft_hi_len(LG), PAD = ifft_pad_a(LG, LGC);
    extern __shared__ __align__(16) float2 ifft_smem[];
    float2* s = ifft_smem;                         // [L + (L >> PAD)][C]
    float2* tw = s + (L + (L >> PAD)) * C;         // [L]
    float2* half = tw + L;                         // [L]
    float2* colt = half + L;                       // [C][W]: hi (HI), lo (32), colw, colg of each column
    constexpr int W = HI + 34;
    const int c = threadIdx.x & (C - 1), t = threadIdx.x >> LGC;
    const long long M = (long long)1 << (LG + lg2);
    const float2* y = Y + (long long)blockIdx.y * ypitch;
    float2* b = B + (long long)blockIdx.y * M;
    const int c0 = blockIdx.x * C;
    // tables first (tw and half are the first 2 L entries of the plan's table, this CTA's columns one run
    // of it: two straight copies, 16 bytes per lane), then the data: the tables land while the data fly
    {
        const float4* g = reinterpret_cast<const float4*>(tab);
        float4* d = reinterpret_cast<float4*>(tw);
        for (int j = threadIdx.x; j < L; j += NT) d[j] = __ldg(g + j);
        const float4* gc = reinterpret_cast<const float4*>(tab + 2 * L + ((size_t)1 << lg2) + (size_t)c0 * W);
        float4* dc = reinterpret_cast<float4*>(colt);
        for (int j = threadIdx.x; j < C * W / 2; j += NT) dc[j] = __ldg(gc + j);
    }
    float2 v[8], m[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const long long k = ((long long)(t + q * T) << lg2) + c0 + c;
        v[q] = y[k];
        m[q] = y[M - k];
    }
    __syncthreads();
    // e^{+2 pi i k / N} = e^{i pi k1 / M1} e^{i pi k2 / M}, k1 = t + q L / 8: half[t] colw[c] times e^{i pi q / 8}
    const float2 w0 = ifft_cmul(half[t], colt[c * W + HI + 32]);
    const float kc[8] = {1.f, 0.92387953251128674f, 0.70710678118654752f, 0.38268343236508977f,
                         0.f, -0.38268343236508977f, -0.70710678118654752f, -0.92387953251128674f};
    const float ks[8] = {0.f, 0.38268343236508977f, 0.70710678118654752f, 0.92387953251128674f,
                         1.f, 0.92387953251128674f, 0.70710678118654752f, 0.38268343236508977f};
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const float2 a = v[q];
        const float2 mc = make_float2(m[q].x, -m[q].y);                  // conj Y[M - k]
        const float2 w = ifft_cmul(w0, make_float2(kc[q], ks[q]));
        const float2 wd = ifft_cmul(w, ifft_sub(a, mc));
        const float2 sum = ifft_add(a, mc);
        v[q] = make_float2(sum.x - wd.y, sum.y + wd.x);                  // sum + i w dif
    }
    // e^{+2 pi i k2 n1 / M} for the outputs n1 = t + r L / 8 in turn: the first from the hi / lo tables, then
    // times colg[c] each
    float2* bc = b + c0 + c;
    // e^{+2 pi i k2 n1 / M} for the outputs n1 = t + r L / 8: a product of two table entries each (ACC), or the
    // first one so and then times colg[c] each
    const float2* ct = colt + c * W;
    float2 pw = ifft_cmul(ct[t >> 5], ct[HI + (t & 31)]);
    const float2 pg = ct[HI + 33];
    ifft_core<LG, LGC, PAD, ACC>(v, s, tw, t, c, t, c, [&](int r, int n1, float2 val) {
        if (ACC) pw = ifft_cmul(ct[n1 >> 5], ct[HI + (n1 & 31)]);
        else if (r > 0) pw = ifft_cmul(pw, pg);
        bc[(long long)n1 << lg2] = ifft_cmul(val, pw);
    });
}

// Pass B.  grid = (M1 / C, rows), CTA = C rows n1 of B x L / 8 threads, L = M2 = 2^LG.
// out: [rows][opitch] floats, the first nout of the 2 M samples.
template <int LG, int LGC, bool ACC>
__global__ void __launch_bounds__(1 << (LG - 3 + LGC), (LG - 3 + LGC) >= 10 ? 1 : IFFT_MINB_B)
k_ifft_pass_b(const float2* __restrict__ B, float* __restrict__ out, long long opitch, long long nout, int lg1,
              float mean, const float2* __restrict__ tab)
{
    constexpr int L = 1 << LG, C = 1 << LGC, T = L / 8, NT = T * C, PAD = ifft_pad_b(LG, LGC);
    extern __shared__ __align__(16) float2 ifft_smem[];
    float2* s = ifft_smem;                         // [L + (L >> PAD)][C]
    float2* tw = s + (L + (L >> PAD)) * C;         // [L]
    // loads (and the first stage) with 8 lanes along a row of B (64-byte runs), the rest and the stores with
    // the lanes across the C rows (runs of 8 C bytes): both sides of the transposition this pass is are
    // then runs of whole sectors
    const int c = threadIdx.x & (C - 1), t = threadIdx.x >> LGC;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int TW = T >= 8 ? T / 8 : 1;         // groups of 8 points along a row
    const int t_in = LG >= 6 ? (warp % TW) * 8 + (lane & 7) : t;
    const int c_in = LG >= 6 ? (warp / TW) * 4 + (lane >> 3) : c;
    const long long M = (long long)1 << (LG + lg1);
    const long long n1 = (long long)blockIdx.x * C + c;
    const float2* b = B + (long long)blockIdx.y * M + (((long long)blockIdx.x * C + c_in) << LG);
    float* o = out + (long long)blockIdx.y * opitch;
    {
        const float4* g = reinterpret_cast<const float4*>(tab + ((size_t)2 << lg1));
        float4* d = reinterpret_cast<float4*>(tw);
        for (int j = threadIdx.x; j < L / 2; j += NT) d[j] = __ldg(g + j);
    }
    float2 v[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) v[q] = b[t_in + q * T];
    __syncthreads();
    // (rows of the caller's array may start on an odd float: then two 4-byte stores per point)
    const bool vec = (reinterpret_cast<uintptr_t>(o) & 7) == 0;
    ifft_core<LG, LGC, PAD, ACC>(v, s, tw, t_in, c_in, t, c, [&](int, int n2, float2 val) {
        const long long n = n1 + ((long long)n2 << lg1);                 // z[n] = (y[2n], y[2n+1])
        if (2 * n + 1 < nout) {
            if (vec) {
                *reinterpret_cast<float2*>(o + 2 * n) = make_float2(val.x + mean, val.y + mean);
            } else {
                o[2 * n] = val.x + mean;
                o[2 * n + 1] = val.y + mean;
            }
        } else if (2 * n < nout) {
            o[2 * n] = val.x + mean;
        }
    });
}

// Pass B with two transforms per thread: a CTA takes 8 rows n1 of B (threads: 4 row pairs x L / 8), so that
// the stores are 64-byte runs (16 bytes per lane) and the loads 64-byte runs of each row.  Tile [rows][8]
// float2, point i in row i + (i >> PAD), PAD = log2 of the first stage's radix: conflict-free for 16-byte
// accesses (enumerated as for ifft_pad_a).
__host__ __device__ constexpr int ifft_pad_b2(int lg) { return lg % 3 ? lg % 3 : 3; }
constexpr size_t ifft_smem_b2(int lg)
{
    return ((size_t)((1 << lg) + ((1 << lg) >> ifft_pad_b2(lg))) * 8 + (size_t)(1 << lg)) * sizeof(float2);
}

template <int LG, bool ACC>
__global__ void __launch_bounds__(1 << (LG - 1), LG >= 11 ? 1 : 2)
k_ifft_pass_b2(const float2* __restrict__ B, float* __restrict__ out, long long opitch, long long nout, int lg1,
               float mean, const float2* __restrict__ tab)
{
    constexpr int L = 1 << LG, T = L / 8, NT = T * 4, PAD = ifft_pad_b2(LG);
    extern __shared__ __align__(16) float2 ifft_smem[];
    float2* s = ifft_smem;                         // [L + (L >> PAD)][8]
    float2* tw = s + (L + (L >> PAD)) * 8;         // [L]
    const int c = threadIdx.x & 3, t = threadIdx.x >> 2;
    const long long M = (long long)1 << (LG + lg1);
    const long long n1 = (long long)blockIdx.x * 8 + 2 * c;
    const float2* b0 = B + (long long)blockIdx.y * M + (n1 << LG);
    float* o = out + (long long)blockIdx.y * opitch;
    {
        const float4* g = reinterpret_cast<const float4*>(tab + ((size_t)2 << lg1));
        float4* d = reinterpret_cast<float4*>(tw);
        for (int j = threadIdx.x; j < L / 2; j += NT) d[j] = __ldg(g + j);
    }
    float2 va[8], vb[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        va[q] = b0[t + q * T];
        vb[q] = b0[L + t + q * T];
    }
    __syncthreads();
    // z[n] = (y[2n], y[2n+1]); this thread's n and n + 1 are 16 contiguous bytes of the row
    const bool vec = (reinterpret_cast<uintptr_t>(o) & 15) == 0;
    ifft_core2<LG, 2, PAD, ACC>(va, vb, s, tw, t, c, [&](int, int n2, float2 a, float2 b) {
        const long long n = n1 + ((long long)n2 << lg1);
        float* p = o + 2 * n;
        if (vec && 2 * n + 3 < nout) {
            *reinterpret_cast<float4*>(p) = make_float4(a.x + mean, a.y + mean, b.x + mean, b.y + mean);
        } else {
            if (2 * n < nout) p[0] = a.x + mean;
            if (2 * n + 1 < nout) p[1] = a.y + mean;
            if (2 * n + 2 < nout) p[2] = b.x + mean;
            if (2 * n + 3 < nout) p[3] = b.y + mean;
        }
    });
}

// M = nfft_out / 2 = M1 M2, both powers of two in [8, 2048]
inline bool ifft_split(long long nfft_out, int* M1, int* M2)
{
    const long long M = nfft_out / 2;
    if (nfft_out < 128 || (M & (M - 1)) != 0) return false;
    int lg = 0;
    while ((1LL << lg) < M) ++lg;
    // (pass A, whose global rows are runs of C elements, takes the shorter factor: 8 columns in 512 threads
    //  up to 512 points; pass B reads whole rows)
    const int l1 = lg / 2, l2 = lg - l1;
    if (l2 > 11 || l1 < 3) return false;
    *M1 = 1 << l1;
    *M2 = 1 << l2;
    return true;
}

// columns side by side in a CTA: 8 (64-byte runs of every global row) up to 512 points, 4 above (CTAs of
// 512 and 1024 threads); FDD_IFFT_WIDE: 8 columns x 1024 points in 1024 threads
inline int ifft_lgc(int lg)
{
    static const bool wide = getenv("FDD_IFFT_WIDE") != nullptr;
    return lg <= 9 ? 3 : (lg == 10 && wide ? 3 : 2);
}

template <int LG, int LGC, bool ACC>
inline int ifft_launch_a(const float2* Y, long long ypitch, float2* B, int lg2, const float2* tab, int rows,
                         cudaStream_t s)
{
    static bool attr = false;
    constexpr size_t bytes = ifft_smem_a(LG, LGC);
    if (!attr) {
        if (cudaFuncSetAttribute(k_ifft_pass_a<LG, LGC, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) !=
            cudaSuccess)
            return -3;
        attr = true;
    }
    k_ifft_pass_a<LG, LGC, ACC><<<dim3((unsigned)((1 << lg2) >> LGC), (unsigned)rows), 1 << (LG - 3 + LGC), bytes, s>>>(
        Y, ypitch, B, lg2, tab);
    return 0;
}

template <int LG, int LGC, bool ACC>
inline int ifft_launch_b(const float2* B, float* out, long long opitch, long long nout, int lg1, float mean,
                         const float2* tab, int rows, cudaStream_t s)
{
    static bool attr = false;
    constexpr size_t bytes = ifft_smem_b(LG, LGC);
    if (!attr) {
        if (cudaFuncSetAttribute(k_ifft_pass_b<LG, LGC, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) !=
            cudaSuccess)
            return -3;
        attr = true;
    }
    k_ifft_pass_b<LG, LGC, ACC><<<dim3((unsigned)((1 << lg1) >> LGC), (unsigned)rows), 1 << (LG - 3 + LGC), bytes, s>>>(
        B, out, opitch, nout, lg1, mean, tab);
    return 0;
}

template <int LG, bool ACC>
inline int ifft_launch_b2(const float2* B, float* out, long long opitch, long long nout, int lg1, float mean,
                          const float2* tab, int rows, cudaStream_t s)
{
    static bool attr = false;
    constexpr size_t bytes = ifft_smem_b2(LG);
    if (!attr) {
        if (cudaFuncSetAttribute(k_ifft_pass_b2<LG, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) !=
            cudaSuccess)
            return -3;
        attr = true;
    }
    k_ifft_pass_b2<LG, ACC><<<dim3((unsigned)((1 << lg1) >> 3), (unsigned)rows), 1 << (LG - 1), bytes, s>>>(
        B, out, opitch, nout, lg1, mean, tab);
    return 0;
}

#define FDD_IFFT_DISPATCH(lg, lgc, CALL)                       \
    switch ((lg) * 4 + (lgc)) {                                \
        case 3 * 4 + 3: { constexpr int LG_ = 3, LGC_ = 3; CALL; break; }   \
        case 4 * 4 + 3: { constexpr int LG_ = 4, LGC_ = 3; CALL; break; }   \
        case 5 * 4 + 3: { constexpr int LG_ = 5, LGC_ = 3; CALL; break; }   \
        case 6 * 4 + 3: { constexpr int LG_ = 6, LGC_ = 3; CALL; break; }   \
        case 7 * 4 + 3: { constexpr int LG_ = 7, LGC_ = 3; CALL; break; }   \
        case 8 * 4 + 3: { constexpr int LG_ = 8, LGC_ = 3; CALL; break; }   \
        case 9 * 4 + 3: { constexpr int LG_ = 9, LGC_ = 3; CALL; break; }   \
        case 10 * 4 + 2: { constexpr int LG_ = 10, LGC_ = 2; CALL; break; } \
        case 10 * 4 + 3: { constexpr int LG_ = 10, LGC_ = 3; CALL; break; } \
        case 11 * 4 + 2: { constexpr int LG_ = 11, LGC_ = 2; CALL; break; } \
        default: rc = -5;                                      \
    }

// the plan's table for nfft_out (ifft_table_elems float2 at tab), made on stream s
inline int ifft_make_tables(long long nfft_out, float2* tab, cudaStream_t s)
{
    int M1, M2;
    if (!ifft_split(nfft_out, &M1, &M2)) return -5;
    int lg1 = 0, lg2 = 0;
    while ((1 << lg1) < M1) ++lg1;
    while ((1 << lg2) < M2) ++lg2;
    const size_t n = ifft_table_elems(lg1, lg2);
    k_ifft_tables<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(tab, lg1, lg2);
    return cudaGetLastError() == cudaSuccess ? 0 : -3;
}

template <bool ACC>
inline int ifft_launch_acc(const float2* Y, long long ypitch, int rows, float* out, long long opitch, long long nout,
                           int lg1, int lg2, float mean, float2* ring, const float2* tab, int batch, cudaStream_t s)
{
    const int lgc1 = ifft_lgc(lg1), lgc2 = ifft_lgc(lg2);
    for (int r0 = 0; r0 < rows; r0 += batch) {
        const int n = rows - r0 < batch ? rows - r0 : batch;
        float2* b = ring;
        int rc = 0;
        FDD_IFFT_DISPATCH(lg1, lgc1,
                          (rc = ifft_launch_a<LG_, LGC_, ACC>(Y + (long long)r0 * ypitch, ypitch, b, lg2, tab, n, s)));
        if (rc != 0) return rc;
        // pass B with two transforms per thread for 2048-point transforms (the paper's 2^23-point series:
        // a5 55.1 ms against 57.8 at 1024 trial DMs; at 1024 points it has fewer instructions and wavefronts
        // but too few warps to hide the exchanges: 19.2 against 18.8 ms, so those keep one per thread)
        float* o = out + (long long)r0 * opitch;
        if (lg2 == 11) rc = ifft_launch_b2<11, ACC>(b, o, opitch, nout, lg1, mean, tab, n, s);
        else
            FDD_IFFT_DISPATCH(lg2, lgc2,
                              (rc = ifft_launch_b<LG_, LGC_, ACC>(b, o, opitch, nout, lg1, mean, tab, n, s)));
        if (rc != 0) return rc;
    }
    return cudaGetLastError() == cudaSuccess ? 0 : -3;
}

// rows of Y -> rows of out, in launches of `batch` rows through the intermediate `ring` ([batch][M] float2);
// accurate: the form with every twiddle from a table (zero-padded series, see ifft_core)
inline int ifft_launch(const float2* Y, long long ypitch, int rows, float* out, long long opitch, long long nout,
                       long long nfft_out, float mean, float2* ring, const float2* tab, int batch, bool accurate,
                       cudaStream_t s)
{
    int M1, M2;
    if (!ifft_split(nfft_out, &M1, &M2)) return -5;
    int lg1 = 0, lg2 = 0;
    while ((1 << lg1) < M1) ++lg1;
    while ((1 << lg2) < M2) ++lg2;
    return accurate ? ifft_launch_acc<true>(Y, ypitch, rows, out, opitch, nout, lg1, lg2, mean, ring, tab, batch, s)
                    : ifft_launch_acc<false>(Y, ypitch, rows, out, opitch, nout, lg1, lg2, mean, ring, tab, batch, s);
}

}  // namespace fdd
