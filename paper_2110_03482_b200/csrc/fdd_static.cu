// fdd_rotate_sum_static (include/fdd.h): step a4 for callers that cannot call cudaMalloc - code under
// CUDA graph capture, tight serving loops, harnesses that forbid allocation.
//
//   Y[j][k] = sum_c X[c][k] * exp(+2 pi i * frac(k * d[j][c] / nfft))      (Eq. 4 + Eq. 7)
//
// A variant of the generic a4 kernel (fdd_kernels_generic.cuh) whose only scratch, the table of 64-bit
// phase steps P[c][j] = frac(d[j][c] / nfft) * 2^64, lives in a file-scope __device__ array instead of
// plan memory: nothing is allocated, here or in a library routine.  The price: a fixed maximum size
// (FDD_STATIC_MAX_PHASES entries = 8 MiB, held by every GPU that loads the library until the process
// exits) and ONE table per device - every call overwrites it, so calls that overlap on the GPU (two
// streams, two host threads) race.
//
// Host code sees g_static_phase only as a stand-in for the symbol, not as a device address: the kernels
// get the address cudaGetSymbolAddress returns, looked up once per device with that device current.
#include "../../include/fdd.h"

#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

// The scratch: file scope, one copy per GPU that loads the library
static __device__ __align__(256) unsigned long long g_static_phase[FDD_STATIC_MAX_PHASES];

namespace {

constexpr int kStaticDT = 8;           // trial DMs per thread (rows of the table are padded to it)
constexpr int kStaticThreads = 128;    // bins per CTA
constexpr int kStaticMaxDevices = 64;

// phase[c][j] for j < ndm_pad: every entry of the part of the table this call uses is written (the
// array keeps the last call's contents), the padding j >= ndm with 0.  delays: [ndm][nchans] samples.
__global__ void __launch_bounds__(256)
k_static_build_phases(const double* __restrict__ delays, int ndm, int nchans, int ndm_pad, double nfft,
                      unsigned long long* __restrict__ phase)
{
    const long long idx = (long long)blockIdx.x * 256 + threadIdx.x;
    if (idx >= (long long)nchans * ndm_pad) return;
    const int c = (int)(idx / ndm_pad), j = (int)(idx - (long long)c * ndm_pad);
    unsigned long long v = 0ULL;
    if (j < ndm) {
        // (nfft a power of two: quotient, fraction and the scaling by 2^64 are all exact in fp64)
        const double cyc = delays[(long long)j * nchans + c] / nfft;
        const double f = cyc - floor(cyc);
        if (f < 1.0) v = __double2ull_rn(f * 18446744073709551616.0);
    }
    phase[idx] = v;
}

// thread = one bin k of kStaticDT trial DMs; a warp covers 32 consecutive bins (coalesced X loads and
// Y stores); CTAs are rasterised DM-tile fastest so that CTAs running together share X through L2
__global__ void __launch_bounds__(kStaticThreads)
k_rotate_sum_static(const float2* __restrict__ X, long long xpitch, const unsigned long long* __restrict__ phase,
                    int ndm_pad, int nchans, long long nbins, int ndm, int n_jtiles, float2* __restrict__ out,
                    float dc_add)
{
    const int jt = blockIdx.x % n_jtiles;
    const long long kt = blockIdx.x / n_jtiles;
    const long long k = kt * kStaticThreads + threadIdx.x;
    const int j0 = jt * kStaticDT;
    const bool live = k < nbins;
    const unsigned int ku = (unsigned int)(live ? k : 0);
    float2 acc[kStaticDT];
#pragma unroll
    for (int i = 0; i < kStaticDT; ++i) acc[i] = make_float2(0.f, 0.f);
    for (int c = 0; c < nchans; ++c) {
        const float2 x = X[(long long)c * xpitch + ku];
        const unsigned long long* prow = phase + (long long)c * ndm_pad + j0;
#pragma unroll
        for (int i = 0; i < kStaticDT; ++i) {
            // k * P mod 2^64 = the fractional cycle of k d / nfft, reduced exactly by integer wrap-around;
            // its top 32 bits as a signed integer are the phase in [-1/2, 1/2) cycles
            const unsigned long long t = prow[i] * (unsigned long long)ku;
            const float cyc = (float)(int)(unsigned int)(t >> 32) * 2.3283064365386963e-10f;   // * 2^-32
            float s, co;
            __sincosf(cyc * 6.283185307179586f, &s, &co);
            acc[i].x = fmaf(x.x, co, acc[i].x);
            acc[i].x = fmaf(-x.y, s, acc[i].x);
            acc[i].y = fmaf(x.x, s, acc[i].y);
            acc[i].y = fmaf(x.y, co, acc[i].y);
        }
    }
    if (!live) return;
#pragma unroll
    for (int i = 0; i < kStaticDT; ++i) {
        const int j = j0 + i;
        if (j >= ndm) break;
        out[(long long)j * nbins + k] = make_float2(acc[i].x + (k == 0 ? dc_add : 0.f), acc[i].y);
    }
}

// device address of g_static_phase on the CURRENT device, looked up once per device
int static_phase_table(unsigned long long** table)
{
    static std::mutex mu;
    static unsigned long long* addr[kStaticMaxDevices] = {};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kStaticMaxDevices) {
        cudaGetLastError();
        return FDD_ERR_CUDA;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        unsigned long long* p = nullptr;
        if (cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_phase) != cudaSuccess || !p) {
            cudaGetLastError();
            return FDD_ERR_CUDA;
        }
        addr[dev] = p;
    }
    *table = addr[dev];
    return FDD_OK;
}

}  // namespace

extern "C" int fdd_rotate_sum_static(const void* x_dev, long long xpitch, const double* delays_dev, int nchans,
                                     long long nbins, long long nfft, int ndm, void* out_dev, float dc_add,
                                     void* cuda_stream)
{
    if (!x_dev || !delays_dev || !out_dev || nchans < 1 || ndm < 1 || nbins < 1 || nfft < 2 ||
        nbins > nfft / 2 + 1 || xpitch < nbins)
        return FDD_ERR_INVALID_ARG;
    const long long ndm_pad = ((long long)ndm + kStaticDT - 1) / kStaticDT * kStaticDT;
    if ((long long)nchans * ndm_pad > (long long)FDD_STATIC_MAX_PHASES) return FDD_ERR_TOO_LARGE;
    const long long n_jt = ndm_pad / kStaticDT;
    const long long n_kt = (nbins + kStaticThreads - 1) / kStaticThreads;
    if (n_jt * n_kt > 2147483647LL) return FDD_ERR_TOO_LARGE;
    unsigned long long* table = nullptr;
    const int rc = static_phase_table(&table);
    if (rc != FDD_OK) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const long long entries = (long long)nchans * ndm_pad;
    k_static_build_phases<<<(unsigned)((entries + 255) / 256), 256, 0, s>>>(delays_dev, ndm, nchans, (int)ndm_pad,
                                                                           (double)nfft, table);
    k_rotate_sum_static<<<(unsigned)(n_jt * n_kt), kStaticThreads, 0, s>>>(
        static_cast<const float2*>(x_dev), xpitch, table, (int)ndm_pad, nchans, nbins, ndm, (int)n_jt,
        static_cast<float2*>(out_dev), dc_add);
    if (cudaGetLastError() != cudaSuccess) return FDD_ERR_CUDA;
    return FDD_OK;
}
