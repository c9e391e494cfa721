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
constexpr int kSym2Depth = 8;          // X prefetch queue depth (channels in flight per thread)

struct Sym2Seed {
    float zrA, ziA, zrB, ziB;
    float2 e0;
    float c2;
};


__device__ __forceinline__ float sym2_rad(unsigned int top)
{
    return (float)(int)top * 1.4629180792671596e-09f;                    // 2 pi * 2^-32
}

// Seed of one (channel, bin) from the phase steps p = (centre A lo, hi, half step lo, hi), each a
// 64-bit binary fraction of a cycle per bin: k * P mod 2^64 is the exact fractional cycle; its
// top 32 bits feed the SFU.  Centre of sub-tile B = centre A + 64 half steps (a carry out of the
// low words is 2^-32 cycle and dropped).  E_0 = (cos, sin) phi, c2 = 2 cos 2 phi.
__device__ __forceinline__ Sym2Seed sym2_seed(float2 x, uint4 p, unsigned int k)
{
    const unsigned int ta = p.y * k + __umulhi(p.x, k);
    const unsigned long long wh = (unsigned long long)p.z * k;
    const unsigned int th = p.w * k + (unsigned int)(wh >> 32);
    const unsigned int tb = ta + __funnelshift_l((unsigned int)wh, th, 6);
    float sa, ca, sb, cb, b0, a0;
    __sincosf(sym2_rad(ta), &sa, &ca);
    __sincosf(sym2_rad(tb), &sb, &cb);
    __sincosf(sym2_rad(th), &b0, &a0);
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

// One channel: 64 accumulate + 15 recurrence FFMA2 with the seed `cur`.
__device__ __forceinline__ void sym2_accumulate(const Sym2Seed& cur, float2 (&UA)[kSymPairs],
                                                float2 (&VA)[kSymPairs], float2 (&UB)[kSymPairs],
                                                float2 (&VB)[kSymPairs])
{
    const float2 zrA = make_float2(cur.zrA, cur.zrA), ziA = make_float2(cur.ziA, cur.ziA);
    const float2 zrB = make_float2(cur.zrB, cur.zrB), ziB = make_float2(cur.ziB, cur.ziB);
    const float2 c2 = make_float2(cur.c2, cur.c2);
    // The recurrence runs one step ahead of the accumulation, so an accumulate FFMA2 never
    // issues right behind the FFMA2 that produces its phasor (that would stall a full FFMA2
    // latency fifteen times per channel).
    float2 ep = make_float2(cur.e0.x, -cur.e0.y);     // E_{-1} = conj(E_0)
    float2 e = cur.e0;                                // E_m
    float2 en = __ffma2_rn(c2, e, make_float2(-ep.x, -ep.y));   // E_{m+1}
#pragma unroll
    for (int m = 0; m < kSymPairs; ++m) {
        float2 enn = en;
        if (m + 2 < kSymPairs) enn = __ffma2_rn(c2, en, make_float2(-e.x, -e.y));   // E_{m+2}
        UA[m] = __ffma2_rn(zrA, e, UA[m]);
        VA[m] = __ffma2_rn(ziA, e, VA[m]);
        UB[m] = __ffma2_rn(zrB, e, UB[m]);
        VB[m] = __ffma2_rn(ziB, e, VB[m]);
        e = en;
        en = enn;
    }
}

__device__ __forceinline__ void sym2_cp_async8(unsigned int saddr, const float2* g)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(saddr), "l"(g) : "memory");
}
__device__ __forceinline__ void sym2_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void sym2_cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ float2 sym2_lds_x(unsigned int addr)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr) : "memory");
    return v;
}

__device__ __forceinline__ uint4 sym2_lds(unsigned int addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}

__global__ void __launch_bounds__(kSym2Threads, 3)
k_rotate_sum_sym2(const float2* __restrict__ X, long long xpitch,
                  const unsigned long long* __restrict__ centre64,
                  const unsigned long long* __restrict__ half64, int nchans, long long nbins,
                  int tile0, int npairs, int ntiles_total, int ndm, float2* __restrict__ out,
                  long long opitch, int row0, float scale, int real_edges, float dc_add)
{
    // Phase steps of the channels in flight, (centre A, half step) per channel.  They are the
    // same for every thread, so they are staged once per CTA: a global load of them inside the
    // channel loop would share a scoreboard with the X prefetch and expose its latency.
    __shared__ uint4 s_p[kSym2Chunk + 2];
    __shared__ float2 s_x[kSym2Depth][kSym2Threads];

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
    unsigned int ku = (unsigned int)k;
    asm volatile("" : "+r"(ku));                      // keep k in a register (no re-derivation)
    const unsigned int sbase = (unsigned int)__cvta_generic_to_shared(s_p);
    const unsigned int xbase = (unsigned int)__cvta_generic_to_shared(&s_x[0][threadIdx.x]);

    // X prefetch queue: every thread streams ITS OWN bin of the next kSym2Depth channels into its
    // own shared-memory slots with cp.async (no thread reads another's slot, so no barrier):
    // registers hold one X value, the queue covers L2 / HBM latency of kSym2Depth iterations.
    const float2* xq = X + k + xpitch;                // next channel to request (1, 2, ...)
    int to_request = nchans - 1;
#pragma unroll
    for (int d = 1; d < kSym2Depth; ++d) {
        if (to_request > 0) sym2_cp_async8(xbase + d * (kSym2Threads * 8), xq);
        sym2_cp_commit();
        xq += xpitch;
        --to_request;
    }

    Sym2Seed cur;
    int slot = 1;                                     // queue slot of channel c + 1
    for (int c0 = 0; c0 < nchans; c0 += kSym2Chunk) {
        const int n = nchans - c0 < kSym2Chunk ? nchans - c0 : kSym2Chunk;
        __syncthreads();
        for (int i = threadIdx.x; i <= n; i += kSym2Threads) {
            const int cc = c0 + i < nchans ? c0 + i : nchans - 1;
            const uint2 a = __ldg(ga + cc), h = __ldg(gh + cc);
            s_p[i] = make_uint4(a.x, a.y, h.x, h.y);
        }
        __syncthreads();
        if (c0 == 0) cur = sym2_seed(X[k], s_p[0], ku);
        unsigned int sp = sbase + 16;                 // table entry of channel c + 1
        for (int i = 0; i < n; ++i) {
            // channel c + kSym2Depth goes into the slot channel c left in the last iteration
            const int wslot = slot == 0 ? kSym2Depth - 1 : slot - 1;
            if (to_request > 0) sym2_cp_async8(xbase + wslot * (kSym2Threads * 8), xq);
            sym2_cp_commit();
            xq += xpitch;
            --to_request;
            sym2_accumulate(cur, UA, VA, UB, VB);     // channel c
            sym2_cp_wait<kSym2Depth - 1>();           // channel c + 1 has landed
            const float2 x1 = sym2_lds_x(xbase + slot * (kSym2Threads * 8));
            cur = sym2_seed(x1, sym2_lds(sp), ku);    // seed of channel c + 1
            sp += 16;
            slot = slot + 1 == kSym2Depth ? 0 : slot + 1;
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
