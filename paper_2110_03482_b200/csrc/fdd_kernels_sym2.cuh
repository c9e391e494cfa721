// Step a4, symmetric kernel with a SHARED recurrence: one CTA tile = NS adjacent 32-DM sub-tiles
// (NS = 3: 96 trial DMs, the default; NS = 2 where that wastes fewer rows) of
// fdd_kernels_sym.cuh's pairing.
//
//   Y[j][k] = sum_c X[c][k] * exp(+2 pi i k d[j][c] / nfft)             (Eq. 4 + Eq. 7,
//                                                                   PAPER.md:64, 82)
//
// When the half DM step h_c is the same in all sub-tiles (a uniform DM grid), the pair phasors
// E_m = (cos, sin)((2m+1) phi), phi = 2 pi k h_c / nfft, are the SAME for all of them; only the
// centre rotation differs:  Z_s = X e^{i theta_s},  theta_s = theta_A + 64 s phi.  Per (channel,
// bin) the kernel then issues 32 NS accumulate FFMA2 (2 per pair, 16 pairs, NS sub-tiles) but
// only 15 recurrence FFMA2, and ONE seed (phase products, table and X loads, c2):
//     NS = 3: 111 FFMA2 per 96 trial DMs = 2.31 FMA lanes per (dm, channel, bin) element,
//             192 accumulator registers, 254 in all, 2 CTAs x 128 threads per SM;
//     NS = 2:  79 FFMA2 per 64 trial DMs = 2.47 lanes, 168 registers, 3 CTAs per SM;
// against 94 FFMA2 per 64 for independent 32-DM tiles.  The recurrence is no longer than before
// (m <= 15), so the error bound of fdd_kernels_sym.cuh is unchanged.  Measured on B200 at
// 1024 channels x 2^20 samples x 4096 trial DMs: NS = 3 183 ms, NS = 2 ~205 ms, 32-DM tiles 333 ms
// (profiles/r01c_*, r01b_*, r01a_*).
#pragma once
#include "fdd_kernels_sym.cuh"

namespace fdd {

constexpr int kSym2Threads = 128;
constexpr int kSym2Chunk = 1024;       // channels whose phase steps are staged in shared memory
constexpr int kSym2Depth = 8;          // X prefetch queue depth (channels in flight per thread)

__device__ __forceinline__ float sym2_rad(unsigned int top)
{
    return (float)(int)top * 1.4629180792671596e-09f;                    // 2 pi * 2^-32
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

template <int NS>
struct Sym2Seed {
    float zr[NS], zi[NS];
    float2 e0;
    float c2;
};

// The three 32-bit phases (fractions of a cycle * 2^32) of one (channel, bin): centre of sub-tile A,
// half step, and 64 half steps (the distance between sub-tile centres), from the staged table
// entry at shared address sp.  Two table formats:
//  kFp64 (nfft <= 2^23): entry = (P_A, P_h, frac(64 P_h)) * 2^(32-pshift) as doubles, P in
//    [-1/2, 1/2) cycles per bin, pshift = max(0, log2 nfft - 21).  The low word of
//    fma(k, P 2^(32-pshift), 1.5 * 2^52) is round(k P 2^(32-pshift)) mod 2^32 (the product stays
//    below 2^51 for k <= nfft/2); shifted left by pshift it is the phase to 2^-(32-pshift) cycle:
//    ONE instruction on the otherwise idle FP64 pipe per phase.  The integer form costs an
//    IMAD.HI/IMAD.WIDE + IMAD per phase in the FMA pipe the accumulation needs (measured:
//    195 -> 186 ms at config 4 / 4096 DMs).
//  !kFp64 (any nfft): entry = (P_A lo, hi, P_h lo, hi), 64-bit binary fractions; k * P mod 2^64
//    by integer multiplies, a carry out of the low words into 64 P_h (2^-32 cycle) dropped.
struct Sym2Phases {
    unsigned int ta, th, step;
};

// kMode 0: FP64-pipe phases, pshift = 0; 1: FP64-pipe phases, pshift > 0; 2: integer phases.
template <int kMode>
__device__ __forceinline__ Sym2Phases sym2_phases(unsigned int sp, unsigned int ku, double kd,
                                                  int pshift)
{
    Sym2Phases ph;
    if (kMode < 2) {
        const double magic = 6755399441055744.0;                         // 1.5 * 2^52
        double pa, p_h, p64h;
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(pa), "=d"(p_h) : "r"(sp));
        asm volatile("ld.shared.f64 %0, [%1+16];" : "=d"(p64h) : "r"(sp));
        const int sh = kMode == 0 ? 0 : pshift;
        ph.ta = (unsigned int)__double2loint(fma(kd, pa, magic)) << sh;
        ph.th = (unsigned int)__double2loint(fma(kd, p_h, magic)) << sh;
        ph.step = (unsigned int)__double2loint(fma(kd, p64h, magic)) << sh;
    } else {
        const uint4 p = sym2_lds(sp);
        ph.ta = p.y * ku + __umulhi(p.x, ku);
        const unsigned long long wh = (unsigned long long)p.z * ku;
        ph.th = p.w * ku + (unsigned int)(wh >> 32);
        ph.step = __funnelshift_l((unsigned int)wh, ph.th, 6);
    }
    return ph;
}

// Seed of one (channel, bin): Z_s = X e^{i theta_s} for the NS sub-tile centres theta_s = theta_A +
// s * (64 half steps), E_0 = (cos, sin) phi, c2 = 2 cos 2 phi from the smaller of |cos|, |sin|
// (2 - 4 sin^2 = 4 cos^2 - 2).  The top 32 bits of each exact fractional cycle feed the SFU.
template <int NS>
__device__ __forceinline__ Sym2Seed<NS> sym2_seed(float2 x, Sym2Phases ph)
{
    const unsigned int ta = ph.ta, th = ph.th, step = ph.step;
    Sym2Seed<NS> s;
    if (NS == 3) {
        // middle sub-tile directly, its neighbours by G^-1 and G = e^{i 64 phi}: 10 FMA-pipe
        // operations and 2 sin/cos pairs instead of 12 and 3
        float sn, cs, gi, gr;
        __sincosf(sym2_rad(ta + step), &sn, &cs);
        __sincosf(sym2_rad(step), &gi, &gr);
        const float z1r = fmaf(x.x, cs, -x.y * sn), z1i = fmaf(x.x, sn, x.y * cs);
        const float t1 = z1i * gi, t2 = z1r * gi;
        s.zr[1] = z1r;
        s.zi[1] = z1i;
        s.zr[2] = fmaf(z1r, gr, -t1);
        s.zi[2] = fmaf(z1i, gr, t2);
        s.zr[0] = fmaf(z1r, gr, t1);
        s.zi[0] = fmaf(z1i, gr, -t2);
    } else {
        unsigned int t = ta;
#pragma unroll
        for (int i = 0; i < NS; ++i) {
            float sn, cs;
            __sincosf(sym2_rad(t), &sn, &cs);
            s.zr[i] = fmaf(x.x, cs, -x.y * sn);
            s.zi[i] = fmaf(x.x, sn, x.y * cs);
            t += step;
        }
    }
    float b0, a0;
    __sincosf(sym2_rad(th), &b0, &a0);
    const float tmin = fminf(fabsf(a0), fabsf(b0));
    const float q = fmaf(-4.f * tmin, tmin, 2.f);
    s.c2 = fabsf(b0) < fabsf(a0) ? q : -q;
    s.e0 = make_float2(a0, b0);
    return s;
}

// One channel: 32 NS accumulate + 15 recurrence FFMA2 with the seed `cur`.  Accumulators as in
// fdd_kernels_sym.cuh but with D_r' = -D_r, so both operands are plain broadcasts:
//        U_m = (S_r, D_i ) += (Z_r, Z_r) * E_m        Y+ = (S_r - D_r', S_i + D_i)
//        V_m = (S_i, D_r') += (Z_i, Z_i) * E_m        Y- = (S_r + D_r', S_i - D_i)
// The recurrence runs one step ahead of the accumulation, so an accumulate FFMA2 never issues
// right behind the FFMA2 that produces its phasor.
template <int NS>
__device__ __forceinline__ void sym2_accumulate(const Sym2Seed<NS>& cur, float2 (&U)[NS][kSymPairs],
                                                float2 (&V)[NS][kSymPairs])
{
    const float2 c2 = make_float2(cur.c2, cur.c2);
    float2 e = cur.e0;                                            // E_m
    float2 en = __ffma2_rn(c2, e, make_float2(-e.x, e.y));        // E_1 = c2 E_0 - conj(E_0)
#pragma unroll
    for (int m = 0; m < kSymPairs; ++m) {
        float2 enn = en;
        if (m + 2 < kSymPairs) enn = __ffma2_rn(c2, en, make_float2(-e.x, -e.y));   // E_{m+2}
#pragma unroll
        for (int i = 0; i < NS; ++i) {
            U[i][m] = __ffma2_rn(make_float2(cur.zr[i], cur.zr[i]), e, U[i][m]);
            V[i][m] = __ffma2_rn(make_float2(cur.zi[i], cur.zi[i]), e, V[i][m]);
        }
        e = en;
        en = enn;
    }
}

// The sub-tiles one launch covers, grouped for the CTAs: group g = sub-tiles tile0 + start[g] ...
// + count[g] - 1 (count <= NS), all continuing one progression.  On a uniform DM grid every group is
// full; on a piecewise-uniform DM plan a group ends where the DM step changes.  Passed by value.
constexpr int kSym2MaxGroups = 256;
struct Sym2Groups {
    unsigned short start[kSym2MaxGroups];
    unsigned char count[kSym2MaxGroups];
};

// kMirror (TIME mode): a CTA holds 64 bins k and their mirrors N/2 - k, and the epilogue writes
// Z[k] = (Y[k] + conj Y[N/2-k]) + i e^{2 pi i k / N} (Y[k] - conj Y[N/2-k]) instead of Y: the inverse
// real transform of N points is then ONE complex transform of N/2 points of Z (its output pairs are
// the even / odd samples), and cuFFT's own pre-processing pass over Y (a quarter of a5) is gone.
template <int NS, int kMinCtas, int kMode, bool kMirror>
__global__ void __launch_bounds__(kSym2Threads, kMinCtas)
k_rotate_sum_sym2(const float2* __restrict__ X, long long xpitch,
                  const unsigned long long* __restrict__ centre64,
                  const unsigned long long* __restrict__ half64, int nchans, long long nbins,
                  int tile0, int ngroups, const Sym2Groups groups, int ndm, float2* __restrict__ out,
                  long long opitch, int row0, float scale, int real_edges, float dc_add,
                  int pshift)
{
    // Phase steps of the channels in flight, (centre A, half step) per channel.  They are the
    // same for every thread, so they are staged once per CTA: a global load of them inside the
    // channel loop would share a scoreboard with the X prefetch and expose its latency.
    __shared__ double4 s_p[kSym2Chunk + 2];         // 32 B per channel, format: sym2_phases
    __shared__ float2 s_x[kSym2Depth][kSym2Threads];

    // 1-D grid, DM tile-group fastest: CTAs resident together read the same X slab through L2.
    const int gr = (int)(blockIdx.x % (unsigned)ngroups);
    const long long kb = blockIdx.x / (unsigned)ngroups;
    bool live;
    long long k;
    if (kMirror) {
        constexpr int kHalf = kSym2Threads / 2;
        const long long H = nbins - 1;                // N/2 (even); pairs (kl, H - kl), kl = 0..H/2
        const long long kl = kb * kHalf + (threadIdx.x & (kHalf - 1));
        const bool upper = threadIdx.x >= kHalf;
        live = upper ? kl < H / 2 : kl <= H / 2;      // the middle bin pairs with itself: lower only
        k = live ? (upper ? H - kl : kl) : H / 2;     // dead lanes redo the middle bin, never stored
    } else {
        const long long kraw = kb * kSym2Threads + threadIdx.x;
        live = kraw < nbins;
        k = live ? kraw : nbins - 1;                  // dead lanes redo the last bin, never stored
    }
    const int tA = tile0 + groups.start[gr];
    const int nsub = groups.count[gr];                // sub-tiles beyond it are computed, not stored

    float2 U[NS][kSymPairs], V[NS][kSymPairs];
#pragma unroll
    for (int i = 0; i < NS; ++i)
#pragma unroll
        for (int m = 0; m < kSymPairs; ++m) U[i][m] = V[i][m] = make_float2(0.f, 0.f);

    const uint2* ga = reinterpret_cast<const uint2*>(centre64 + (size_t)tA * nchans);
    const uint2* gh = reinterpret_cast<const uint2*>(half64 + (size_t)tA * nchans);
    const double kd = (double)k;
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

    Sym2Seed<NS> cur;
    int slot = 1;                                     // queue slot of channel c + 1
    for (int c0 = 0; c0 < nchans; c0 += kSym2Chunk) {
        const int n = nchans - c0 < kSym2Chunk ? nchans - c0 : kSym2Chunk;
        __syncthreads();
        for (int i = threadIdx.x; i <= n; i += kSym2Threads) {
            const int cc = c0 + i < nchans ? c0 + i : nchans - 1;
            const uint2 a = __ldg(ga + cc), h = __ldg(gh + cc);
            if (kMode < 2) {
                const unsigned long long ua = ((unsigned long long)a.y << 32) | a.x;
                const unsigned long long uh = ((unsigned long long)h.y << 32) | h.x;
                // signed 64-bit fractions of a cycle (wrap = reduction to [-1/2, 1/2)) times
                // 2^-(32+pshift)
                const double sc = __hiloint2double((1023 - 32 - pshift) << 20, 0);
                s_p[i] = make_double4((double)(long long)ua * sc, (double)(long long)uh * sc,
                                      (double)(long long)(uh << 6) * sc, 0.0);
            } else {
                *reinterpret_cast<uint4*>(&s_p[i]) = make_uint4(a.x, a.y, h.x, h.y);
            }
        }
        __syncthreads();
        if (c0 == 0) cur = sym2_seed<NS>(X[k], sym2_phases<kMode>(sbase, ku, kd, pshift));
        unsigned int sp = sbase + 32;                 // table entry of channel c + 1
        for (int i = 0; i < n; ++i) {
            const int wslot = slot == 0 ? kSym2Depth - 1 : slot - 1;
            if (to_request > 0) sym2_cp_async8(xbase + wslot * (kSym2Threads * 8), xq);
            sym2_cp_commit();
            xq += xpitch;
            --to_request;
            sym2_accumulate<NS>(cur, U, V);           // channel c
            sym2_cp_wait<kSym2Depth - 1>();           // channel c + 1 has landed
            const float2 x1 = sym2_lds_x(xbase + slot * (kSym2Threads * 8));
            cur = sym2_seed<NS>(x1, sym2_phases<kMode>(sp, ku, kd, pshift));   // seed of channel c + 1
            sp += 32;
            slot = slot + 1 == kSym2Depth ? 0 : slot + 1;
        }
    }
    const bool edge = real_edges && (k == 0 || k == nbins - 1);
    const float dc = k == 0 ? dc_add : 0.f;           // the mean a2 removed (already scaled)
    if (!kMirror) {
        if (!live) return;
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            if (s >= nsub) break;
            const int j0 = (tA + s) * kSymT;
#pragma unroll
            for (int m = 0; m < kSymPairs; ++m) {
                const float2 u = U[s][m], v = V[s][m];
                const int jp = j0 + kSymPairs + m, jm = j0 + kSymPairs - 1 - m;
                if (jp < ndm)
                    out[(long long)(jp - row0) * opitch + k] =
                        make_float2((u.x - v.y) * scale + dc, edge ? 0.f : (v.x + u.y) * scale);
                if (jm < ndm)
                    out[(long long)(jm - row0) * opitch + k] =
                        make_float2((u.x + v.y) * scale + dc, edge ? 0.f : (v.x - u.y) * scale);
            }
        }
        return;
    }

    // Mirror epilogue: partners (threads t and t ^ 64) swap their Y through shared memory, 16 rows
    // at a time, and each writes Z of its own bin (bin N/2 itself has no Z entry).
    constexpr int kHalf = kSym2Threads / 2;
    const long long H = nbins - 1;
    float2* ex = reinterpret_cast<float2*>(s_p);      // [kSymPairs][kSym2Threads], after the loop
    double wsd, wcd;
    sincospi((double)k / (double)H, &wsd, &wcd);      // w = e^{2 pi i k / N}, N = 2 H
    const float ws = (float)wsd, wc = (float)wcd;
    const bool self = (k == H - k);
    const bool store = live && k < H;
    __syncthreads();                                  // everyone is done with s_p
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        if (s >= nsub) break;                         // (uniform over the CTA)
        const int j0 = (tA + s) * kSymT;
#pragma unroll
        for (int sgn = 0; sgn < 2; ++sgn) {
            float2 y[kSymPairs];
#pragma unroll
            for (int m = 0; m < kSymPairs; ++m) {
                const float2 u = U[s][m], v = V[s][m];
                y[m] = sgn == 0 ? make_float2((u.x - v.y) * scale + dc, edge ? 0.f : (v.x + u.y) * scale)
                                : make_float2((u.x + v.y) * scale + dc, edge ? 0.f : (v.x - u.y) * scale);
                ex[m * kSym2Threads + threadIdx.x] = y[m];
            }
            __syncthreads();
#pragma unroll
            for (int m = 0; m < kSymPairs; ++m) {
                const int j = sgn == 0 ? j0 + kSymPairs + m : j0 + kSymPairs - 1 - m;
                float2 p = ex[m * kSym2Threads + (threadIdx.x ^ kHalf)];     // Y[N/2 - k]
                if (self) p = y[m];
                // A = Y[k], B = conj(Y[N/2 - k]):  Z = (A + B) + i w (A - B)
                const float sr = y[m].x + p.x, si = y[m].y - p.y;
                const float dr = y[m].x - p.x, di = y[m].y + p.y;
                const float2 z = make_float2(sr - (wc * di + ws * dr), si + (wc * dr - ws * di));
                if (store && j < ndm) out[(long long)(j - row0) * opitch + k] = z;
            }
            __syncthreads();
        }
    }
}

// Greedy grouping of sub-tiles [tile0, tile0 + ntl) into runs of at most ns that continue one
// progression; returns the number of groups (starts relative to tile0).
inline int sym2_group(const SymTables& t, int tile0, int ntl, int ns, std::vector<unsigned short>* start,
                      std::vector<unsigned char>* count)
{
    start->clear();
    count->clear();
    for (int i = 0; i < ntl;) {
        int n = 1;
        while (n < ns && i + n < ntl && t.cont[tile0 + i + n - 1]) ++n;
        start->push_back((unsigned short)i);
        count->push_back((unsigned char)n);
        i += n;
    }
    return (int)start->size();
}

// The launch shape of rows [j_begin, j_begin + rows): sub-tiles per CTA group (NS) and the group
// lists, one per launch of at most kSym2MaxGroups groups.  Made once per chunk at plan time /
// first use and kept by the plan, so a launch allocates nothing.
struct Sym2Shape {
    int ns = 3;
    std::vector<Sym2Groups> groups;
    std::vector<int> ngroups;
};

inline Sym2Shape sym2_shape(const SymTables& t, int j_begin, int rows)
{
    Sym2Shape sh;
    const int tile0 = j_begin / kSymT;
    const int ntl = (rows + kSymT - 1) / kSymT;
    std::vector<unsigned short> gs3, gs2;
    std::vector<unsigned char> gc3, gc2;
    // 96-DM groups (NS = 3) unless 64-DM groups leave fewer sub-tiles idle: measured cost of one
    // group per (channel, warp): 294 cycles for NS = 3, 232 for NS = 2
    const long long cost3 = 294LL * sym2_group(t, tile0, ntl, 3, &gs3, &gc3);
    const long long cost2 = 232LL * sym2_group(t, tile0, ntl, 2, &gs2, &gc2);
    sh.ns = cost3 <= cost2 ? 3 : 2;
    const std::vector<unsigned short>& gs = sh.ns == 3 ? gs3 : gs2;
    const std::vector<unsigned char>& gc = sh.ns == 3 ? gc3 : gc2;
    const int all = (int)gs.size();
    for (int g0 = 0; g0 < all; g0 += kSym2MaxGroups) {
        const int n = all - g0 < kSym2MaxGroups ? all - g0 : kSym2MaxGroups;
        Sym2Groups g;
        for (int i = 0; i < kSym2MaxGroups; ++i) {
            g.start[i] = i < n ? gs[g0 + i] : 0;
            g.count[i] = i < n ? gc[g0 + i] : 0;
        }
        sh.groups.push_back(g);
        sh.ngroups.push_back(n);
    }
    return sh;
}

// Rows [j_begin, j_begin + rows) -> dst[(j - j_begin) * opitch + k]; j_begin a multiple of kSymT.
template <int NS, int kMinCtas>
inline int sym2_launch(const Sym2Shape& sh, bool mirror, long long nfft, const SymTables& t, const float2* X,
                       long long xpitch, int nchans, long long nbins, int ndm, int j_begin, int rows,
                       float2* dst, long long opitch, float scale, int real_edges, float dc_add,
                       cudaStream_t s)
{
    if (j_begin % kSymT != 0 || !t.centre64 || sh.ns != NS) return -5;
    const int tile0 = j_begin / kSymT;
    const int ntl = (rows + kSymT - 1) / kSymT;
    if (ntl > 65535) return -5;
    const int row_end = j_begin + rows < ndm ? j_begin + rows : ndm;
    // mirror: 64 bin pairs (k, N/2 - k), k = 0 .. N/4, per CTA
    const long long nkb = mirror ? ((nbins - 1) / 2 + 1 + kSym2Threads / 2 - 1) / (kSym2Threads / 2)
                                 : (nbins + kSym2Threads - 1) / kSym2Threads;
    int pshift = 0;                                   // FP64-pipe phases: see sym2_phases
    while ((nfft >> pshift) > (1LL << 21)) ++pshift;
    const int mode = pshift == 0 ? 0 : (pshift <= 2 ? 1 : 2);   // nfft <= 2^23; longer: integer phases
#define FDD_SYM2_LAUNCH(MODE, MIRROR)                                                              \
    k_rotate_sum_sym2<NS, kMinCtas, MODE, MIRROR><<<grid, kSym2Threads, 0, s>>>(                   \
        X, xpitch, t.centre64, t.half64, nchans, nbins, tile0, ngroups, groups, row_end, dst,      \
        opitch, j_begin, scale, real_edges, dc_add, pshift)
    for (size_t l = 0; l < sh.groups.size(); ++l) {                // one launch per 256 groups
        const int ngroups = sh.ngroups[l];
        const Sym2Groups& groups = sh.groups[l];
        if ((long long)ngroups * nkb > 2147483647LL) return -5;
        const unsigned grid = (unsigned)(ngroups * nkb);
        if (mirror) {
            if (mode == 0) FDD_SYM2_LAUNCH(0, true);
            else if (mode == 1) FDD_SYM2_LAUNCH(1, true);
            else FDD_SYM2_LAUNCH(2, true);
        } else {
            if (mode == 0) FDD_SYM2_LAUNCH(0, false);
            else if (mode == 1) FDD_SYM2_LAUNCH(1, false);
            else FDD_SYM2_LAUNCH(2, false);
        }
    }
#undef FDD_SYM2_LAUNCH
    return cudaGetLastError() == cudaSuccess ? 0 : -3;
}

}  // namespace fdd
