// C ABI of the FDD hot path (include/fdd.h): plan tables, scratch, cuFFT plans, stage launches.
// Everything numerical on the device happens in the kernels of fdd_kernels_*.cuh and in cuFFT
// (allowed for the FFT stages); the host only builds the phase tables.
#include "../../include/fdd.h"

#include <cuda_runtime.h>
#include <cufft.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <map>
#include <new>
#include <utility>
#include <vector>

#include "fdd_kernels_generic.cuh"
#include "fdd_kernels_ifft.cuh"
#include "fdd_kernels_krec.cuh"
#include "fdd_kernels_pad.cuh"
#include "fdd_kernels_pre.cuh"
#include "fdd_kernels_sym.cuh"
#include "fdd_kernels_sym2.cuh"
#include "fdd_kernels_tc.cuh"
#include "fdd_kernels_tdd.cuh"

namespace {

constexpr double kDefaultKdm = 4.148808e3;            // MHz^2 pc^-1 cm^3 s (reading S5)
constexpr long long kPitchAlign = 16;                 // float2 elements (128 B)
constexpr size_t kYBudgetBytes = (size_t)24 << 30;    // TIME-mode Y scratch per DM chunk
// ... of a plan on the tensor-core kernel, whose cost is per launch, not per row (measured at the
// paper's shape, 1024 channels x 2^23 points x 1024 trial DMs: one launch 219 ms, three 384-row chunks
// 660 ms, the FP32 kernel 377 ms): room for 2048 rows of 2^23 points
constexpr size_t kYBudgetTensorBytes = ((size_t)64 << 30) + ((size_t)1 << 27);
constexpr int kC2RBatch = 384;                        // rows per cuFFT inverse call (4 x 96-DM groups)
constexpr int kHostChunkRows = kC2RBatch;             // fdd_execute_host: DM rows per pipelined chunk
constexpr int kHostRingChunks = 3;                    // fdd_execute_host: output chunks resident on the device
// Rows per launch of the own inverse: its intermediate takes 512 MiB (128 rows at nfft = 2^20; launches of
// fewer rows leave SMs idle at their tails: 23.2 ms with 16 rows, 20.5 with 128 at 4096 x 2^20), at
// least 8 and at most 512 rows.  FDD_IFFT_BATCH overrides (experiments).
int ifft_batch(long long nfft_out)
{
    static const int env = [] {
        const char* e = getenv("FDD_IFFT_BATCH");
        const int v = e ? atoi(e) : 0;
        return v >= 1 && v <= 4096 ? v : 0;
    }();
    if (env) return env;
    const long long rows = (1LL << 26) / (nfft_out / 2 > 0 ? nfft_out / 2 : 1);
    return rows < 8 ? 8 : (rows > 512 ? 512 : (int)rows);
}
// AUTO: launches with fewer trial DMs take the FP32 kernels.  Measured on B200 (1024 channels x 2^20
// samples): the tensor-core kernel's 64-row form costs 26.9 ms for any number of trial DMs up to 1024,
// the shared-recurrence kernel 25.9 ms at 512 and 47 ms at 1024 (proportional to the rows).
constexpr int kTensorMinRows = 640;

inline long long round_up(long long a, long long b) { return (a + b - 1) / b * b; }

struct StageEvent {
    int stage;
    cudaEvent_t beg, end;
};

}  // namespace

struct fdd_plan {
    // problem
    int nchans = 0, ndm = 0;
    long long nsamps = 0, nfft = 0, nbins = 0;
    // output side: reduced-length inverse FFT (fdd_plan_set_decimation); = input side
    // sizes when log2_dec == 0
    int log2_dec = 0;
    long long nfft_out = 0, nbins_out = 0, nsamps_out = 0;
    double tsamp = 0, f_lo = 0, f_hi = 0, kdm = kDefaultKdm;
    bool from_delays = false;
    std::vector<double> dm_list;
    std::vector<double> delays;          // [ndm][nchans], samples
    double max_delay = 0;
    long long valid_len = 0;
    int device = 0;
    int num_sms = 0;
    float offset = 0.f;                  // subtracted by a2, restored in bin 0 by a4 (S21)
    // zero-padded series (fdd_kernels_pad.cuh): the rectangle's share of the lowest bins, per plan
    bool padded = false;
    int pad_k = 0;                       // bins treated exactly
    float2* pad_tab = nullptr;           // [ndm][pad_k], built by fdd_plan_prepare / on first use
    bool pad_ready = false;
    // device buffers
    float2* X = nullptr;                 // [nchans][xpitch] spectra
    float* xreal = nullptr;              // [nchans][nfft] unpacked series (out-of-place R2C input)
    bool r2c_inplace = false;            // large plans: the series are unpacked into X's rows instead
    long long xpitch = 0;
    float2* Y = nullptr;                 // TIME mode: [y_rows][ypitch] (lazily allocated)
    long long ypitch = 0;
    int y_rows = 0;
    unsigned long long* phase64 = nullptr;   // generic kernel: [nchans][ndm_pad]
    // bin-recurrence kernel (nfft <= 2^23): the same fractions as doubles * 2^(32 - pshift), and
    // the per-bin phasor step exp(2 pi i frac(d / nfft)); [nchans][ndm_pad] each
    double* rec_p32 = nullptr;
    float2* rec_step = nullptr;
    int rec_pshift = -1;                     // -1: series too long, generic kernel only
    bool rec_ready = false;
    std::vector<double> rec_p32_host;        // plan-owned upload buffers (asynchronous copies read them)
    std::vector<float2> rec_step_host;
    int ndm_pad = 0;
    size_t y_budget = 0;                     // TIME-mode Y scratch budget in bytes (fdd_plan_set_y_budget)
    // a4 launch shapes of the shared-recurrence kernel, made once per (first row, rows) chunk
    std::map<std::pair<int, int>, fdd::Sym2Shape> sym2_shapes;
    fdd::SymTables sym;                  // symmetric kernel tables (device) + tiling
    bool sym_ok = false;
    int kernel = FDD_KERNEL_GENERIC;     // resolved choice
    int kernel_request = FDD_KERNEL_AUTO;
    // FFT
    cufftHandle r2c = 0;
    bool have_r2c = false;
    // a5 plans in two families: [0] C2R of nfft_out points from Y; [1] C2C of nfft_out/2 points from
    // the pre-twiddled Z the mirrored sym2 epilogue writes (fdd_kernels_sym2.cuh, kMirror)
    cufftHandle c2r[2] = {0, 0}, c2r_tail[2] = {0, 0};
    bool have_c2r[2] = {false, false}, have_c2r_tail[2] = {false, false};
    int c2r_batch = 0, c2r_tail_batch = 0;
    void* fft_ws = nullptr;
    size_t fft_ws_bytes = 0;
    // a5 by the hand-written two-pass transform (fdd_kernels_ifft.cuh) instead of cuFFT
    int inverse_request = FDD_INVERSE_AUTO;
    bool ifft_on = false;                // decided with the TIME-mode resources
    bool dc_in_bin0 = true;              // a4 restores the mean in bin 0 (false: the own inverse adds it)
    float2* ifft_ring = nullptr;         // [ifft_batch(nfft_out)][nfft_out / 2]
    size_t ifft_ring_bytes = 0;
    float2* ifft_tab = nullptr;          // the own inverse's twiddle tables (fdd_kernels_ifft.cuh)
    size_t ifft_tab_bytes = 0;
    bool ifft_no_room = false;           // AUTO: the intermediate did not fit, this plan stays on cuFFT
    // multi-beam execution (fdd_execute_beams): spectra and TIME-mode sums of one group of beams
    float2* beam_X = nullptr;            // [beam_group][nchans][xpitch]
    float2* beam_Y = nullptr;            // [beam_group][ndm][ypitch]
    int beam_group = 0;
    // host staging (fdd_execute_host)
    unsigned char* stage_in = nullptr;
    void* stage_out = nullptr;
    size_t stage_out_bytes = 0;
    cudaStream_t copy_stream = nullptr;
    std::vector<cudaEvent_t> chunk_events;
    std::vector<cudaEvent_t> in_events;
    // profiling
    bool profiling = false;
    std::vector<StageEvent> events;
    size_t events_used = 0;
    int launches[FDD_NUM_STAGES] = {0, 0, 0, 0, 0, 0};
    // time-domain comparator (fdd_tdd_execute), built on first use
    unsigned char* tdd_xt = nullptr;     // [nchans][tdd_tpitch] transposed bytes, periodic tail
    long long tdd_tpitch = 0;
    int* tdd_shifts = nullptr;           // [nchans][ndm_pad] shifts mod nsamps
    size_t scratch_bytes = 0;
};

namespace {

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard()
    {
        int cur = -1;
        if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
    }
};

template <class T>
int dev_alloc(fdd_plan* p, T** ptr, size_t count)
{
    void* v = nullptr;
    const size_t bytes = count * sizeof(T);
    if (cudaMalloc(&v, bytes ? bytes : 1) != cudaSuccess) {
        cudaGetLastError();
        return FDD_ERR_ALLOC;
    }
    *ptr = static_cast<T*>(v);
    p->scratch_bytes += bytes;
    return FDD_OK;
}

// a1: delay table from frequencies and DMs (Eq. 1), in long double.
void build_delays(fdd_plan* p)
{
    p->delays.assign((size_t)p->ndm * p->nchans, 0.0);
    const long double fhi = p->f_hi;
    for (int c = 0; c < p->nchans; ++c) {
        const long double nu =
            p->nchans == 1 ? fhi
                           : (long double)p->f_lo +
                                 (long double)c * ((long double)p->f_hi - (long double)p->f_lo) /
                                     (long double)(p->nchans - 1);
        const long double per_dm =
            (long double)p->kdm * (1.0L / (nu * nu) - 1.0L / (fhi * fhi)) / (long double)p->tsamp;
        for (int j = 0; j < p->ndm; ++j)
            p->delays[(size_t)j * p->nchans + c] = (double)((long double)p->dm_list[j] * per_dm);
    }
}

void finish_delay_stats(fdd_plan* p)
{
    double m = 0;
    for (double d : p->delays) m = fmax(m, fabs(d));
    p->max_delay = m;
    // S10: mathematically integer delays may evaluate a hair above the integer
    p->valid_len = p->nsamps - (long long)ceil(m * (1.0 - 1e-12));
    if (p->valid_len < 0) p->valid_len = 0;          // delays longer than the series: nothing is valid
}

// The tensor-core kernel needs ONE arithmetic progression over all trial DMs (a uniform DM grid), at
// most 1024 channels (phase steps staged in shared memory) and nfft <= 2^23 (FP64-pipe phases).
bool tensor_ok(const fdd_plan* p)
{
    return p->sym_ok && p->sym.pair_ok && p->nchans <= fdd::kTcMaxChans && p->rec_pshift >= 0;
}

// AUTO: the fastest kernel the delay table allows.
int resolve_kernel(const fdd_plan* p, int request)
{
    const bool sym2_ok = p->sym_ok;      // groups of sub-tiles follow the DM plan's uniform segments
    const bool any_ap = p->sym.nap > 0;
    switch (request) {
        case FDD_KERNEL_TENSOR: return tensor_ok(p) ? FDD_KERNEL_TENSOR : FDD_KERNEL_GENERIC;
        case FDD_KERNEL_GENERIC: return FDD_KERNEL_GENERIC;
        case FDD_KERNEL_SYMMETRIC: return p->sym_ok ? FDD_KERNEL_SYMMETRIC : FDD_KERNEL_GENERIC;
        case FDD_KERNEL_SYMMETRIC2: return sym2_ok ? FDD_KERNEL_SYMMETRIC2 : FDD_KERNEL_GENERIC;
        case FDD_KERNEL_MIXED: return sym2_ok ? FDD_KERNEL_SYMMETRIC2
                                              : (any_ap ? FDD_KERNEL_MIXED : FDD_KERNEL_GENERIC);
        default:
            // measured on B200 (1024 channels x 2^20 samples): the tensor-core kernel costs 27 ms up to
            // 1024 trial DMs per launch, 36 ms up to 2048 and 46 ms up to 4096, the shared-recurrence
            // kernel 46 ms per 1024 trial DMs
            if (tensor_ok(p) && p->ndm >= kTensorMinRows) return FDD_KERNEL_TENSOR;
            if (sym2_ok) return FDD_KERNEL_SYMMETRIC2;
            // a few tiles hold a change of DM step: those rows alone take the generic kernel
            return 2 * p->sym.nap >= p->sym.ntiles && any_ap ? FDD_KERNEL_MIXED : FDD_KERNEL_GENERIC;
    }
}

int upload_generic_table(fdd_plan* p)
{
    std::vector<unsigned long long> tab((size_t)p->nchans * p->ndm_pad, 0ULL);
    for (int j = 0; j < p->ndm; ++j)
        for (int c = 0; c < p->nchans; ++c)
            tab[(size_t)c * p->ndm_pad + j] = fdd::sym_fixed64(
                (long double)p->delays[(size_t)j * p->nchans + c] / (long double)p->nfft);
    // (a cudaMemcpy from pageable memory returns once the data are staged; the synchronize makes
    // sure they have landed before a kernel on a non-blocking stream can read them)
    if (cudaMemcpy(p->phase64, tab.data(), tab.size() * sizeof(unsigned long long),
                   cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaDeviceSynchronize() != cudaSuccess) {
        cudaGetLastError();
        return FDD_ERR_CUDA;
    }
    p->pad_ready = false;
    p->rec_ready = false;                // rebuilt by fdd_plan_prepare / the next generic launch
    p->sym2_shapes.clear();
    return FDD_OK;
}

// Tables of the bin-recurrence kernel (plans on uniform DM grids never need them): the same
// fractions frac(d / nfft) as doubles * 2^(32 - pshift), and exp(2 pi i frac).  Made by
// fdd_plan_prepare, or by the first generic launch of a plan that was not prepared: then the
// device buffers are allocated here (cudaMalloc may synchronise) and the upload is queued on the
// launching stream from plan-owned host buffers, in order with the kernel that reads them.
int ensure_rec_tables(fdd_plan* p, cudaStream_t s)
{
    if (p->rec_ready) return FDD_OK;
    const size_t n = (size_t)p->nchans * p->ndm_pad;
    int rc;
    if (!p->rec_p32 && (rc = dev_alloc(p, &p->rec_p32, n)) != FDD_OK) return rc;
    if (!p->rec_step && (rc = dev_alloc(p, &p->rec_step, n)) != FDD_OK) return rc;
    // (the host buffers may still feed an earlier upload of a plan whose k_dm was changed)
    if (cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); return FDD_ERR_CUDA; }
    p->rec_p32_host.assign(n, 0.0);
    p->rec_step_host.assign(n, make_float2(1.f, 0.f));
    const long double two_pi = 6.283185307179586476925286766559L;
    for (int j = 0; j < p->ndm; ++j)
        for (int c = 0; c < p->nchans; ++c) {
            const unsigned long long f = fdd::sym_fixed64(
                (long double)p->delays[(size_t)j * p->nchans + c] / (long double)p->nfft);
            const long double cyc = (long double)(long long)f * 5.42101086242752217e-20L;   // [-1/2, 1/2)
            const size_t i = (size_t)c * p->ndm_pad + j;
            p->rec_p32_host[i] = (double)ldexpl(cyc, 32 - p->rec_pshift);
            p->rec_step_host[i] = make_float2((float)cosl(two_pi * cyc), (float)sinl(two_pi * cyc));
        }
    if (cudaMemcpyAsync(p->rec_p32, p->rec_p32_host.data(), n * sizeof(double), cudaMemcpyHostToDevice,
                        s) != cudaSuccess ||
        cudaMemcpyAsync(p->rec_step, p->rec_step_host.data(), n * sizeof(float2),
                        cudaMemcpyHostToDevice, s) != cudaSuccess) {
        cudaGetLastError();
        return FDD_ERR_CUDA;
    }
    p->rec_ready = true;
    return FDD_OK;
}

int build_tables(fdd_plan* p)
{
    finish_delay_stats(p);
    int rc = upload_generic_table(p);
    if (rc != FDD_OK) return rc;
    rc = fdd::sym_build_tables(&p->sym, p->delays.data(), p->ndm, p->nchans, p->nfft, &p->sym_ok,
                               &p->scratch_bytes);
    if (rc != FDD_OK) return rc;
    p->kernel = resolve_kernel(p, p->kernel_request);
    return FDD_OK;
}

int make_fft_plans(fdd_plan* p)
{
    // R2C, out of place (cuFFT's in-place form adds a packing pass: 6.8 vs 5.1 ms at 1024 x 2^20):
    // real rows of pitch nfft floats in xreal, complex rows of pitch xpitch in X.
    size_t ws_r2c = 0;
    if (cufftCreate(&p->r2c) != CUFFT_SUCCESS) return FDD_ERR_CUFFT;
    p->have_r2c = true;
    if (cufftSetAutoAllocation(p->r2c, 0) != CUFFT_SUCCESS) return FDD_ERR_CUFFT;
    long long n[1] = {p->nfft};
    // (in place, for plans whose unpacked copy alone would take 16 GiB - the paper's 2^23-point series:
    //  real rows of pitch 2 xpitch floats inside X's own rows)
    const long long rpitch = p->r2c_inplace ? 2 * p->xpitch : p->nfft;
    long long inembed[1] = {rpitch}, onembed[1] = {p->xpitch};
    if (cufftMakePlanMany64(p->r2c, 1, n, inembed, 1, rpitch, onembed, 1, p->xpitch,
                            CUFFT_R2C, p->nchans, &ws_r2c) != CUFFT_SUCCESS)
        return FDD_ERR_CUFFT;
    p->fft_ws_bytes = ws_r2c;
    return FDD_OK;
}

int make_c2r_plan(fdd_plan* p, int family, cufftHandle* h, int batch, size_t* ws)
{
    if (cufftCreate(h) != CUFFT_SUCCESS) return FDD_ERR_CUFFT;
    if (cufftSetAutoAllocation(*h, 0) != CUFFT_SUCCESS) return FDD_ERR_CUFFT;
    const bool direct = (p->nsamps_out == p->nfft_out);     // straight into the caller's rows
    long long inembed[1] = {p->ypitch};
    if (family == 0) {
        long long n[1] = {p->nfft_out};
        long long onembed[1] = {direct ? p->nfft_out : 2 * p->ypitch};
        const long long odist = direct ? p->nfft_out : 2 * p->ypitch;
        if (cufftMakePlanMany64(*h, 1, n, inembed, 1, p->ypitch, onembed, 1, odist, CUFFT_C2R, batch,
                                ws) != CUFFT_SUCCESS)
            return FDD_ERR_CUFFT;
    } else {
        // nfft_out / 2 complex points; the output pairs are the even / odd real samples
        long long n[1] = {p->nfft_out / 2};
        long long onembed[1] = {direct ? p->nfft_out / 2 : p->ypitch};
        const long long odist = direct ? p->nfft_out / 2 : p->ypitch;
        if (cufftMakePlanMany64(*h, 1, n, inembed, 1, p->ypitch, onembed, 1, odist, CUFFT_C2C, batch,
                                ws) != CUFFT_SUCCESS)
            return FDD_ERR_CUFFT;
    }
    return FDD_OK;
}

// The a5 family the plan's kernel feeds: 1 = the half-length complex inverse of the pre-twiddled
// spectrum the mirrored sym2 epilogue writes, 0 = cuFFT's C2R from Y.
int time_family(const fdd_plan* p)
{
    // (a zero-padded plan adds the rectangle's table to Y after a4, so a4 must write plain sums; the
    //  hand-written inverse forms the half-length spectrum itself)
    int m1, m2;
    if (p->inverse_request == FDD_INVERSE_TWO_PASS && fdd::ifft_split(p->nfft_out, &m1, &m2)) return 0;
    return (p->kernel == FDD_KERNEL_SYMMETRIC2 && p->nfft_out >= 4 && !p->padded) ? 1 : 0;
}

void drop_c2r_plan(cufftHandle* h, bool* have)
{
    if (*have) cufftDestroy(*h);
    *have = false;
}

// TIME-mode resources (a FOURIER-only plan such as config 5 never needs the 16 GiB of Y): made by
// fdd_plan_prepare(TIME), or by the first TIME execute of a plan that was not prepared.
int ensure_time_resources(fdd_plan* p, int family)
{
    int rc;
    if (!p->Y) {
        p->ypitch = round_up(p->nbins_out, kPitchAlign);
        const size_t row_bytes = (size_t)p->ypitch * sizeof(float2);
        const size_t budget = p->y_budget ? p->y_budget
                                          : (p->kernel == FDD_KERNEL_TENSOR ? kYBudgetTensorBytes : kYBudgetBytes);
        long long rows = (long long)(budget / row_bytes);
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) {
            long long fit = (long long)(free_b / 2 / row_bytes);
            if (fit < rows) rows = fit;
        }
        // DM chunks: whole cuFFT batches (4 x 96-DM groups) if possible, else whole 96-DM groups,
        // else whole 32-DM tiles, else multiples of 8 (the generic kernels' DM tile)
        if (rows >= p->ndm) rows = p->ndm;
        else rows = rows >= kC2RBatch ? rows / kC2RBatch * kC2RBatch
                                      : (rows >= 96 ? rows / 96 * 96 : (rows >= 32 ? 32 : rows / 8 * 8));
        if (rows < 1) return FDD_ERR_ALLOC;
        p->y_rows = (int)rows;
        int batch = kC2RBatch;
        if (const char* e = getenv("FDD_C2R_BATCH")) { const int v = atoi(e); if (v > 0) batch = v; }
        p->c2r_batch = p->y_rows < batch ? p->y_rows : batch;
        // tails: of a full Y chunk and of the last (short) chunk; at most one distinct tail size
        const int last_rows = p->ndm % p->y_rows ? p->ndm % p->y_rows : p->y_rows;
        int tail = last_rows % p->c2r_batch;
        if (tail == 0) tail = p->y_rows % p->c2r_batch;
        p->c2r_tail_batch = tail;
        if ((rc = dev_alloc(p, &p->Y, (size_t)p->y_rows * p->ypitch)) != FDD_OK) return rc;
    }
    if (p->have_c2r[family]) return FDD_OK;
    size_t ws_a = 0, ws_b = 0;
    rc = make_c2r_plan(p, family, &p->c2r[family], p->c2r_batch, &ws_a);
    p->have_c2r[family] = true;                  // (the handle exists; dropped below on failure)
    if (rc == FDD_OK && p->c2r_tail_batch) {
        rc = make_c2r_plan(p, family, &p->c2r_tail[family], p->c2r_tail_batch, &ws_b);
        p->have_c2r_tail[family] = true;
    }
    const size_t need = ws_a > ws_b ? ws_a : ws_b;
    if (rc == FDD_OK && need > p->fft_ws_bytes) {
        // (no execute is in flight on a plan that is being grown: plans are not re-entrant)
        if (cudaDeviceSynchronize() != cudaSuccess) rc = FDD_ERR_CUDA;
        if (rc == FDD_OK) {
            if (p->fft_ws) { cudaFree(p->fft_ws); p->scratch_bytes -= p->fft_ws_bytes; p->fft_ws = nullptr; }
            p->fft_ws_bytes = 0;
            rc = dev_alloc(p, reinterpret_cast<unsigned char**>(&p->fft_ws), need);
            if (rc == FDD_OK) p->fft_ws_bytes = need;
        }
    }
    // every plan works in the one shared area (never two transforms in flight)
    if (rc == FDD_OK && cufftSetWorkArea(p->r2c, p->fft_ws) != CUFFT_SUCCESS) rc = FDD_ERR_CUFFT;
    for (int f = 0; f < 2 && rc == FDD_OK; ++f) {
        if (p->have_c2r[f] && cufftSetWorkArea(p->c2r[f], p->fft_ws) != CUFFT_SUCCESS) rc = FDD_ERR_CUFFT;
        if (p->have_c2r_tail[f] && cufftSetWorkArea(p->c2r_tail[f], p->fft_ws) != CUFFT_SUCCESS)
            rc = FDD_ERR_CUFFT;
    }
    if (rc != FDD_OK) {
        // a half-made handle must not survive: the next execute starts this family from scratch
        drop_c2r_plan(&p->c2r[family], &p->have_c2r[family]);
        drop_c2r_plan(&p->c2r_tail[family], &p->have_c2r_tail[family]);
    }
    return rc;
}

void drop_time_resources(fdd_plan* p)
{
    for (int f = 0; f < 2; ++f) {
        drop_c2r_plan(&p->c2r[f], &p->have_c2r[f]);
        drop_c2r_plan(&p->c2r_tail[f], &p->have_c2r_tail[f]);
    }
    if (p->Y) {
        cudaFree(p->Y);
        p->scratch_bytes -= (size_t)p->y_rows * p->ypitch * sizeof(float2);
        p->Y = nullptr;
    }
    if (p->beam_Y) {
        cudaFree(p->beam_Y);
        p->scratch_bytes -= (size_t)p->beam_group * p->ndm * p->ypitch * sizeof(float2);
        p->beam_Y = nullptr;
    }
    if (p->ifft_ring) {
        cudaFree(p->ifft_ring);
        p->scratch_bytes -= p->ifft_ring_bytes;
        p->ifft_ring = nullptr;
        p->ifft_ring_bytes = 0;
    }
    if (p->ifft_tab) {
        cudaFree(p->ifft_tab);
        p->scratch_bytes -= p->ifft_tab_bytes;
        p->ifft_tab = nullptr;
        p->ifft_tab_bytes = 0;
    }
    p->ifft_on = false;
    p->ifft_no_room = false;
    p->y_rows = 0;
    p->c2r_tail_batch = 0;
    p->sym2_shapes.clear();
}

// Both TIME-mode families a chunked run may need (a Y chunk off the 32-DM tiling falls back to
// cuFFT's C2R); returns the family to use.
int ensure_time_family(fdd_plan* p, int* family_out)
{
    int family = time_family(p);
    int rc = ensure_time_resources(p, family);
    if (rc != FDD_OK) return rc;
    if (p->kernel == FDD_KERNEL_TENSOR && p->kernel_request == FDD_KERNEL_AUTO && p->y_rows < p->ndm &&
        p->y_rows < kTensorMinRows) {
        // The sums of all trial DMs do not fit the Y scratch and a chunk is shorter than the tensor-core
        // kernel pays for (its cost does not depend on the rows of a launch): this plan stays on the
        // FP32 kernel, whose cost is proportional to the rows (the paper's 2^23-point series at 4096 DMs).
        p->kernel = FDD_KERNEL_SYMMETRIC2;
        family = time_family(p);
        if ((rc = ensure_time_resources(p, family)) != FDD_OK) return rc;
    }
    if (family == 1 && p->y_rows < p->ndm && p->y_rows % fdd::kSymT != 0) {
        family = 0;                          // chunks off the 32-DM tiling run the generic kernel
        if ((rc = ensure_time_resources(p, family)) != FDD_OK) return rc;
    }
    *family_out = family;
    int m1, m2;
    // AUTO: the own inverse where a4 writes plain sums (measured faster than cuFFT's C2R there), unless
    // its intermediate does not fit
    const bool want = p->inverse_request == FDD_INVERSE_TWO_PASS || p->inverse_request == FDD_INVERSE_AUTO;
    p->ifft_on = family == 0 && want && !p->ifft_no_room && fdd::ifft_split(p->nfft_out, &m1, &m2);
    if (p->ifft_on && !p->ifft_ring) {
        const size_t n = (size_t)ifft_batch(p->nfft_out) * (size_t)(p->nfft_out / 2);
        rc = dev_alloc(p, &p->ifft_ring, n);
        if (rc != FDD_OK && p->inverse_request == FDD_INVERSE_AUTO) {
            p->ifft_on = false;                  // no room for the intermediate: cuFFT
            p->ifft_no_room = true;
            return FDD_OK;
        }
        if (rc != FDD_OK) return rc;
        p->ifft_ring_bytes = n * sizeof(float2);
    }
    if (p->ifft_on && !p->ifft_tab) {
        int l1 = 0, l2 = 0;
        while ((1 << l1) < m1) ++l1;
        while ((1 << l2) < m2) ++l2;
        const size_t n = fdd::ifft_table_elems(l1, l2);
        if ((rc = dev_alloc(p, &p->ifft_tab, n)) != FDD_OK) return rc;
        p->ifft_tab_bytes = n * sizeof(float2);
        // (made on the default stream; synchronised so that an execute on any stream finds it)
        if (fdd::ifft_make_tables(p->nfft_out, p->ifft_tab, nullptr) != 0 || cudaDeviceSynchronize() != cudaSuccess) {
            cudaGetLastError();
            return FDD_ERR_CUDA;
        }
    }
    return FDD_OK;
}

void destroy_plan(fdd_plan* p)
{
    if (!p) return;
    DeviceGuard g(p->device);
    cudaDeviceSynchronize();
    if (p->have_r2c) cufftDestroy(p->r2c);
    for (int f = 0; f < 2; ++f) {
        if (p->have_c2r[f]) cufftDestroy(p->c2r[f]);
        if (p->have_c2r_tail[f]) cufftDestroy(p->c2r_tail[f]);
    }
    cudaFree(p->X);
    cudaFree(p->xreal);
    cudaFree(p->tdd_xt);
    cudaFree(p->tdd_shifts);
    cudaFree(p->Y);
    cudaFree(p->phase64);
    cudaFree(p->rec_p32);
    cudaFree(p->rec_step);
    cudaFree(p->fft_ws);
    cudaFree(p->stage_in);
    cudaFree(p->stage_out);
    cudaFree(p->pad_tab);
    cudaFree(p->ifft_ring);
    cudaFree(p->ifft_tab);
    cudaFree(p->beam_X);
    cudaFree(p->beam_Y);
    fdd::sym_free_tables(&p->sym);
    for (auto& e : p->events) { cudaEventDestroy(e.beg); cudaEventDestroy(e.end); }
    for (auto& e : p->chunk_events) cudaEventDestroy(e);
    for (auto& e : p->in_events) cudaEventDestroy(e);
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    cudaGetLastError();
    delete p;
}

int create_common(fdd_plan* p)
{
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return FDD_ERR_CUDA; }
    if (cudaGetDevice(&p->device) != cudaSuccess) return FDD_ERR_CUDA;
    if (cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, p->device) != cudaSuccess)
        return FDD_ERR_CUDA;
    p->nfft = 2;
    while (p->nfft < p->nsamps) p->nfft <<= 1;
    p->nbins = p->nfft / 2 + 1;
    p->nfft_out = p->nfft; p->nbins_out = p->nbins; p->nsamps_out = p->nsamps;
    // The mean of unsigned-byte data stays out of the fp32 transforms.  Without zero padding it lives in
    // bin 0 alone; with padding it is a rectangle, handled in fdd_kernels_pad.cuh.
    p->offset = 128.f;
    p->padded = p->nsamps != p->nfft;
    p->pad_k = (int)(p->nbins < fdd::kPadExactBins ? p->nbins : fdd::kPadExactBins);
    p->xpitch = round_up(p->nbins, kPitchAlign);
    p->ndm_pad = (int)round_up(p->ndm, fdd::kGenDT);
    int rc = dev_alloc(p, &p->X, (size_t)p->nchans * p->xpitch);
    if (rc != FDD_OK) return rc;
    p->r2c_inplace = (size_t)p->nchans * (size_t)p->nfft * sizeof(float) >= ((size_t)16 << 30);
    if (const char* e = getenv("FDD_R2C_INPLACE")) p->r2c_inplace = atoi(e) != 0;     // (tests)
    if (!p->r2c_inplace) {
        rc = dev_alloc(p, &p->xreal, (size_t)p->nchans * p->nfft);
        if (rc != FDD_OK) return rc;
    }
    rc = dev_alloc(p, &p->phase64, (size_t)p->nchans * p->ndm_pad);
    if (rc != FDD_OK) return rc;
    p->rec_pshift = 0;
    while ((p->nfft >> p->rec_pshift) > (1LL << 21)) ++p->rec_pshift;
    if (p->rec_pshift > 2) p->rec_pshift = -1;           // > 2^23 points: integer phases only
    rc = build_tables(p);
    if (rc != FDD_OK) return rc;
    rc = make_fft_plans(p);
    if (rc != FDD_OK) return rc;
    if (p->fft_ws_bytes) {
        size_t need = p->fft_ws_bytes;
        p->fft_ws_bytes = 0;
        rc = dev_alloc(p, reinterpret_cast<unsigned char**>(&p->fft_ws), need);
        if (rc != FDD_OK) return rc;
        p->fft_ws_bytes = need;
    }
    if (cufftSetWorkArea(p->r2c, p->fft_ws) != CUFFT_SUCCESS) return FDD_ERR_CUFFT;
    return FDD_OK;
}

// ---- profiling helpers -----------------------------------------------------------------
struct StageTimer {
    fdd_plan* p;
    cudaStream_t s;
    StageEvent* cur = nullptr;
    StageTimer(fdd_plan* plan, cudaStream_t stream) : p(plan), s(stream) {}
    void begin(int stage, int launches)
    {
        p->launches[stage] += launches;
        if (!p->profiling) return;
        if (p->events_used == p->events.size()) {
            StageEvent e;
            e.stage = stage;
            if (cudaEventCreate(&e.beg) != cudaSuccess || cudaEventCreate(&e.end) != cudaSuccess) {
                cudaGetLastError();
                return;
            }
            p->events.push_back(e);
        }
        cur = &p->events[p->events_used++];
        cur->stage = stage;
        cudaEventRecord(cur->beg, s);
    }
    void end()
    {
        if (cur) cudaEventRecord(cur->end, s);
        cur = nullptr;
    }
};

// time tiles [tile0, tile0 + ntiles) of 64 samples (ntiles < 0: all of them)
// xdst: the spectra buffer the R2C of this series will write (its rows hold the series first when the
// plan transforms in place)
int launch_unpack(fdd_plan* p, const unsigned char* in_u8, cudaStream_t s, long long tile0 = 0,
                  long long ntiles = -1, float2* xdst = nullptr)
{
    if (ntiles < 0) ntiles = (p->nfft + fdd::kUnpackTile - 1) / fdd::kUnpackTile;
    if (ntiles == 0) return FDD_OK;
    dim3 grid((unsigned)ntiles, (unsigned)((p->nchans + fdd::kUnpackTile - 1) / fdd::kUnpackTile));
    float* xf = p->r2c_inplace ? reinterpret_cast<float*>(xdst ? xdst : p->X) : p->xreal;
    const long long rpitch = p->r2c_inplace ? 2 * p->xpitch : p->nfft;
    const bool vec = (p->nchans % 4 == 0) && ((uintptr_t)in_u8 % 4 == 0);
    if (vec)
        fdd::k_unpack_transpose<4><<<grid, 256, 0, s>>>(in_u8, xf, p->nchans, p->nsamps, p->nfft,
                                                        rpitch, p->offset, tile0);
    else
        fdd::k_unpack_transpose<1><<<grid, 256, 0, s>>>(in_u8, xf, p->nchans, p->nsamps, p->nfft,
                                                        rpitch, p->offset, tile0);
    return cudaGetLastError() == cudaSuccess ? FDD_OK : FDD_ERR_CUDA;
}

// Zero-padded plans: the per-plan table of fdd_kernels_pad.cuh (fp64 on the device, once per plan).
int ensure_pad_table(fdd_plan* p, cudaStream_t s)
{
    if (!p->padded || p->pad_ready) return FDD_OK;
    int rc;
    if (!p->pad_tab && (rc = dev_alloc(p, &p->pad_tab, (size_t)p->ndm * p->pad_k)) != FDD_OK) return rc;
    dim3 grid((unsigned)((p->pad_k + 127) / 128), (unsigned)p->ndm);
    fdd::k_pad_build_table<<<grid, 128, 0, s>>>(p->phase64, p->ndm_pad, p->nchans, p->ndm, p->pad_k, p->nsamps,
                                                p->nfft, (double)p->offset, p->pad_tab);
    if (cudaGetLastError() != cudaSuccess) return FDD_ERR_CUDA;
    p->pad_ready = true;
    return FDD_OK;
}

// after a3: the rectangle's spectrum goes back into the bins where it is no larger than the data
int launch_pad_add_rect(fdd_plan* p, float2* X, cudaStream_t s)
{
    if (!p->padded || p->pad_k >= p->nbins) return FDD_OK;
    dim3 grid((unsigned)((p->nbins - p->pad_k + 255) / 256), (unsigned)((p->nchans + 31) / 32));
    fdd::k_pad_add_rect<<<grid, 256, 0, s>>>(X, p->xpitch, p->nchans, p->pad_k, p->nbins, p->nsamps, p->nfft,
                                             (double)p->offset);
    return cudaGetLastError() == cudaSuccess ? FDD_OK : FDD_ERR_CUDA;
}

// after a4: ... and into the lowest bins of the sums, from the table
int launch_pad_add_table(fdd_plan* p, int j_begin, int rows, float2* dst, long long opitch, int mode,
                         cudaStream_t s)
{
    if (!p->padded) return FDD_OK;
    int rc = ensure_pad_table(p, s);
    if (rc != FDD_OK) return rc;
    const int kuse = (int)(p->pad_k < p->nbins_out ? p->pad_k : p->nbins_out);
    const float scale = mode == FDD_MODE_TIME ? (float)(1.0 / (double)p->nfft) : 1.0f;
    for (int r0 = 0; r0 < rows; r0 += 32768) {
        const int n = rows - r0 < 32768 ? rows - r0 : 32768;
        dim3 grid((unsigned)((kuse + 255) / 256), (unsigned)n);
        fdd::k_pad_add_table<<<grid, 256, 0, s>>>(dst + (long long)r0 * opitch, opitch, p->pad_tab, p->pad_k, kuse,
                                                  j_begin + r0, n, scale, mode == FDD_MODE_TIME ? 1 : 0,
                                                  p->nbins_out);
    }
    return cudaGetLastError() == cudaSuccess ? FDD_OK : FDD_ERR_CUDA;
}

// a4 on DM rows [j_begin, j_begin + rows) into dst (row pitch opitch float2).
// mirror (SYMMETRIC2, TIME mode only): dst receives the pre-twiddled Z of the half-length inverse
// transform instead of Y (fdd_kernels_sym2.cuh).
int launch_rotate_sum_kernel(fdd_plan* p, int kernel, int j_begin, int rows, float2* dst,
                             long long opitch, int mode, cudaStream_t s, bool mirror)
{
    const float scale = mode == FDD_MODE_TIME ? (float)(1.0 / (double)p->nfft) : 1.0f;
    const int real_edges = mode == FDD_MODE_TIME ? 1 : 0;      // reading S8
    // bin 0 of every trial DM gets back the mean a2 removed: offset * nchans * nsamps (* scale)
    const double dc_raw = p->padded ? 0.0 : (double)p->offset * (double)p->nchans * (double)p->nsamps;
    const bool dc_in_bin0 = p->dc_in_bin0;
    const float dc_add = mode == FDD_MODE_TIME ? (dc_in_bin0 ? (float)(dc_raw / (double)p->nfft) : 0.f) : (float)dc_raw;
    // (AUTO sends short chunks to the FP32 kernel; an explicit FDD_KERNEL_TENSOR request does not)
    if (kernel == FDD_KERNEL_TENSOR && j_begin % fdd::kSymT == 0 && !mirror &&
        rows >= (p->kernel_request == FDD_KERNEL_TENSOR ? 1 : kTensorMinRows)) {
        // fp16 operands: X times a power of two such that |X| <= 255 nsamps cannot overflow them
        int e = 0;
        frexp((p->padded ? 256.0 : 128.0) * (double)p->nsamps, &e);      // |X| < 2^e
        const float xscale = (float)ldexp(1.0, 15 - e);
        const int per = fdd::kTcT * (fdd::kTcRows / 2);                          // trial DMs per launch
        for (int r0 = 0; r0 < rows; r0 += per) {
            const int n = rows - r0 < per ? rows - r0 : per;
            const int rc = fdd::tc_launch(p->sym, p->nfft, p->X, p->xpitch, p->nchans, p->nbins_out, p->ndm,
                                          j_begin + r0, n, dst + (long long)r0 * opitch, opitch, scale,
                                          real_edges, dc_add, xscale, p->num_sms, s);
            if (rc != 0) return rc;
        }
        return FDD_OK;
    }
    if (kernel == FDD_KERNEL_TENSOR) kernel = FDD_KERNEL_SYMMETRIC2;   // (a short chunk, or one off the 32-DM tiling)
    if (kernel == FDD_KERNEL_SYMMETRIC2 && j_begin % fdd::kSymT == 0) {
        // the grouping of the chunk's 32-DM sub-tiles is made once per (first row, rows)
        auto it = p->sym2_shapes.find(std::make_pair(j_begin, rows));
        if (it == p->sym2_shapes.end())
            it = p->sym2_shapes.emplace(std::make_pair(j_begin, rows),
                                        fdd::sym2_shape(p->sym, j_begin, rows)).first;
        const fdd::Sym2Shape& sh = it->second;
        if (sh.ns == 3)
            return fdd::sym2_launch<3, 2>(sh, mirror, p->nfft, p->sym, p->X, p->xpitch, p->nchans, p->nbins_out,
                                          p->ndm, j_begin, rows, dst, opitch, scale, real_edges, dc_add, s);
        return fdd::sym2_launch<2, 3>(sh, mirror, p->nfft, p->sym, p->X, p->xpitch, p->nchans, p->nbins_out,
                                      p->ndm, j_begin, rows, dst, opitch, scale, real_edges, dc_add, s);
    }
    // (a chunk that does not start on a 32-DM tile - only with rows of > 0.75 GiB - goes generic)
    if ((kernel == FDD_KERNEL_SYMMETRIC || kernel == FDD_KERNEL_SYMMETRIC2) &&
        j_begin % fdd::kSymT == 0)
        return fdd::sym_launch(p->sym, p->X, p->xpitch, p->nchans, p->nbins_out, p->ndm, j_begin, rows,
                               dst, opitch, scale, real_edges, dc_add, s);
    const int n_jt = (rows + fdd::kGenDT - 1) / fdd::kGenDT;
    if (p->rec_pshift >= 0 && j_begin % fdd::kRecDT == 0) {
        // any delay table, phasors by recurrence along the bins (fdd_kernels_krec.cuh)
        const int rcs = ensure_rec_tables(p, s);
        if (rcs != FDD_OK) return rcs;
        const long long per_cta = (long long)fdd::kRecThreads * fdd::kRecL;
        const long long n_kt = (p->nbins_out + per_cta - 1) / per_cta;
        if ((long long)n_jt * n_kt > 2147483647LL) return FDD_ERR_UNSUPPORTED;
        fdd::k_rotate_sum_krec<<<(unsigned)(n_jt * n_kt), fdd::kRecThreads, 0, s>>>(
            p->X, p->xpitch, p->rec_p32, p->rec_step, p->ndm_pad, p->nchans, p->nbins_out, j_begin + rows,
            j_begin, n_jt, dst, opitch, scale, real_edges, dc_add, p->rec_pshift);
        return cudaGetLastError() == cudaSuccess ? FDD_OK : FDD_ERR_CUDA;
    }
    const long long n_kt = (p->nbins_out + fdd::kGenThreads - 1) / fdd::kGenThreads;
    if ((long long)n_jt * n_kt > 2147483647LL) return FDD_ERR_UNSUPPORTED;
    fdd::k_rotate_sum_generic<<<(unsigned)(n_jt * n_kt), fdd::kGenThreads, 0, s>>>(
        p->X, p->xpitch, p->phase64, p->ndm_pad, p->nchans, p->nbins_out, j_begin + rows, j_begin, n_jt,
        dst, opitch, scale, real_edges, dc_add);
    return cudaGetLastError() == cudaSuccess ? FDD_OK : FDD_ERR_CUDA;
}

// a4 with the plan's kernel; FDD_KERNEL_MIXED: runs of 32-DM tiles that are arithmetic progressions
// take the shared-recurrence kernel, the tiles in between (a change of DM step inside them) the
// generic one.
int launch_rotate_sum_plain(fdd_plan* p, int j_begin, int rows, float2* dst, long long opitch, int mode,
                            cudaStream_t s, bool mirror);

int launch_rotate_sum(fdd_plan* p, int j_begin, int rows, float2* dst, long long opitch, int mode,
                      cudaStream_t s, bool mirror = false)
{
    const int rc = launch_rotate_sum_plain(p, j_begin, rows, dst, opitch, mode, s, mirror);
    if (rc != FDD_OK) return rc;
    return launch_pad_add_table(p, j_begin, rows, dst, opitch, mode, s);
}

int launch_rotate_sum_plain(fdd_plan* p, int j_begin, int rows, float2* dst, long long opitch, int mode,
                            cudaStream_t s, bool mirror)
{
    if (p->kernel != FDD_KERNEL_MIXED || j_begin % fdd::kSymT != 0)
        return launch_rotate_sum_kernel(p, p->kernel == FDD_KERNEL_MIXED ? FDD_KERNEL_GENERIC : p->kernel,
                                        j_begin, rows, dst, opitch, mode, s, mirror);
    const int t0 = j_begin / fdd::kSymT, t1 = (j_begin + rows + fdd::kSymT - 1) / fdd::kSymT;
    for (int t = t0; t < t1;) {
        const bool ap = p->sym.ap[t] != 0;
        int e = t + 1;
        while (e < t1 && (p->sym.ap[e] != 0) == ap) ++e;
        const int jb = t * fdd::kSymT;
        const int je = e * fdd::kSymT < j_begin + rows ? e * fdd::kSymT : j_begin + rows;
        const int rc = launch_rotate_sum_kernel(p, ap ? FDD_KERNEL_SYMMETRIC2 : FDD_KERNEL_GENERIC, jb,
                                                je - jb, dst + (long long)(jb - j_begin) * opitch,
                                                opitch, mode, s, false);
        if (rc != FDD_OK) return rc;
        t = e;
    }
    return FDD_OK;
}

int launch_c2r_rows(fdd_plan* p, int family, int rows, float2* ysrc, float* dst, cudaStream_t s,
                    int* launches)
{
    // ysrc: [rows][ypitch]; dst: caller rows (pitch nsamps).
    if (p->ifft_on && family == 0) {
        // the mean a2 removed comes back here, after the transform (not zero padded: a constant)
        const float mean = p->padded ? 0.f
                                     : (float)((double)p->offset * (double)p->nchans * (double)p->nsamps / (double)p->nfft);
        const int rc = fdd::ifft_launch(ysrc, p->ypitch, rows, dst, p->nsamps_out, p->nsamps_out, p->nfft_out, mean,
                                        p->ifft_ring, p->ifft_tab, ifft_batch(p->nfft_out), p->padded, s);
        *launches += 2 * ((rows + ifft_batch(p->nfft_out) - 1) / ifft_batch(p->nfft_out));
        return rc == 0 ? FDD_OK : (rc == -5 ? FDD_ERR_UNSUPPORTED : FDD_ERR_CUDA);
    }
    const bool direct = (p->nsamps_out == p->nfft_out);
    int done = 0;
    while (done < rows) {
        int left = rows - done;
        cufftHandle h;
        int b;
        if (left >= p->c2r_batch) { h = p->c2r[family]; b = p->c2r_batch; }
        else if (p->have_c2r_tail[family] && left >= p->c2r_tail_batch) { h = p->c2r_tail[family]; b = p->c2r_tail_batch; }
        else return FDD_ERR_UNSUPPORTED;     // cannot happen: tails are planned in ensure_time_resources
        if (cufftSetStream(h, s) != CUFFT_SUCCESS) return FDD_ERR_CUFFT;
        float2* src = ysrc + (long long)done * p->ypitch;
        float* drow = dst + (long long)done * p->nsamps_out;
        if (direct) {
            if ((family == 0 ? cufftExecC2R(h, src, drow)
                             : cufftExecC2C(h, src, reinterpret_cast<float2*>(drow), CUFFT_INVERSE)) !=
                CUFFT_SUCCESS)
                return FDD_ERR_CUFFT;
            ++*launches;
        } else {
            if ((family == 0 ? cufftExecC2R(h, src, reinterpret_cast<float*>(src))
                             : cufftExecC2C(h, src, src, CUFFT_INVERSE)) != CUFFT_SUCCESS)
                return FDD_ERR_CUFFT;
            if (cudaMemcpy2DAsync(dst + (long long)done * p->nsamps_out, (size_t)p->nsamps_out * sizeof(float),
                                  src, (size_t)p->ypitch * sizeof(float2),
                                  (size_t)p->nsamps_out * sizeof(float), b, cudaMemcpyDeviceToDevice,
                                  s) != cudaSuccess)
                return FDD_ERR_CUDA;
            *launches += 2;
        }
        done += b;
    }
    return FDD_OK;
}

int check_plan(const fdd_plan* p) { return p ? FDD_OK : FDD_ERR_INVALID_ARG; }

// Stages a2+a3.
int run_pre(fdd_plan* p, const unsigned char* in_u8, cudaStream_t s, StageTimer& tm, bool unpacked = false)
{
    int rc = FDD_OK;
    if (!unpacked) {
        tm.begin(FDD_STAGE_UNPACK, 1);
        rc = launch_unpack(p, in_u8, s);
        tm.end();
    }
    if (rc != FDD_OK) return rc;
    tm.begin(FDD_STAGE_R2C, 1);
    if (cufftSetStream(p->r2c, s) != CUFFT_SUCCESS) return FDD_ERR_CUFFT;
    if (cufftExecR2C(p->r2c, p->r2c_inplace ? reinterpret_cast<float*>(p->X) : p->xreal, p->X) != CUFFT_SUCCESS)
        return FDD_ERR_CUFFT;
    const int rcp = launch_pad_add_rect(p, p->X, s);
    tm.end();
    return rcp;
}

// Stages a4+a5 from the spectra in p->X.  chunk_done (optional) is called after each DM chunk
// has been queued, with (j_begin, rows), so fdd_execute_host can overlap the copy back.
// chunk_rows > 0 caps the DM rows per chunk (multiple of kC2RBatch), for copy/compute overlap.
// ring_rows > 0 (a multiple of chunk_rows): `out` is a ring of that many rows, DM row j lands in
// ring row j % ring_rows, and chunk_begin(j_begin) is called before a chunk's work is queued so
// the caller can make the stream wait until the ring slot has been drained.
template <class F, class G>
int run_post(fdd_plan* p, void* out, int mode, cudaStream_t s, StageTimer& tm, F chunk_done,
             int chunk_rows, int ring_rows, G chunk_begin)
{
    auto out_row = [&](int j0) { return (long long)(ring_rows > 0 ? j0 % ring_rows : j0); };
    if (mode == FDD_MODE_FOURIER) {
        const int step = chunk_rows > 0 ? chunk_rows : p->ndm;
        for (int j0 = 0; j0 < p->ndm; j0 += step) {
            const int rows = (p->ndm - j0 < step) ? p->ndm - j0 : step;
            chunk_begin(j0);
            tm.begin(FDD_STAGE_ROTATE_SUM, 1);
            int rc = launch_rotate_sum(p, j0, rows, static_cast<float2*>(out) + out_row(j0) * p->nbins_out,
                                       p->nbins_out, mode, s);
            tm.end();
            if (rc != FDD_OK) return rc;
            chunk_done(j0, rows);
        }
        return FDD_OK;
    }
    // SYMMETRIC2 writes the pre-twiddled spectrum of the half-length complex inverse (family 1)
    int family = 0;
    int rc = ensure_time_family(p, &family);
    if (rc != FDD_OK) return rc;
    const int step = (chunk_rows > 0 && chunk_rows < p->y_rows) ? chunk_rows : p->y_rows;
    for (int j0 = 0; j0 < p->ndm; j0 += step) {
        const int rows = (p->ndm - j0 < step) ? p->ndm - j0 : step;
        chunk_begin(j0);
        tm.begin(FDD_STAGE_ROTATE_SUM, 1);
        p->dc_in_bin0 = !p->ifft_on;
        rc = launch_rotate_sum(p, j0, rows, p->Y, p->ypitch, mode, s, family == 1);
        p->dc_in_bin0 = true;
        tm.end();
        if (rc != FDD_OK) return rc;
        int nl = 0;
        tm.begin(FDD_STAGE_C2R, 0);
        rc = launch_c2r_rows(p, family, rows, p->Y, static_cast<float*>(out) + out_row(j0) * p->nsamps_out,
                             s, &nl);
        tm.end();
        p->launches[FDD_STAGE_C2R] += nl;
        if (rc != FDD_OK) return rc;
        chunk_done(j0, rows);
    }
    return FDD_OK;
}

void reset_profile(fdd_plan* p)
{
    p->events_used = 0;
    for (int i = 0; i < FDD_NUM_STAGES; ++i) p->launches[i] = 0;
}

}  // namespace

extern "C" {

int fdd_plan_create(fdd_plan** plan_out, int nchans, long long nsamps, double tsamp_s,
                    double f_lo_mhz, double f_hi_mhz, const double* dm_list_host, int ndm)
{
    if (!plan_out) return FDD_ERR_INVALID_ARG;
    *plan_out = nullptr;
    if (nchans < 1 || nsamps < 2 || !(tsamp_s > 0) || !(f_lo_mhz > 0) || !(f_hi_mhz >= f_lo_mhz) ||
        !isfinite(tsamp_s) || !isfinite(f_hi_mhz) || ndm < 1 || !dm_list_host)
        return FDD_ERR_INVALID_ARG;
    for (int j = 0; j < ndm; ++j)
        if (!isfinite(dm_list_host[j])) return FDD_ERR_INVALID_ARG;
    fdd_plan* p = new (std::nothrow) fdd_plan();
    if (!p) return FDD_ERR_ALLOC;
    p->nchans = nchans; p->nsamps = nsamps; p->tsamp = tsamp_s;
    p->f_lo = f_lo_mhz; p->f_hi = f_hi_mhz; p->ndm = ndm;
    p->dm_list.assign(dm_list_host, dm_list_host + ndm);
    build_delays(p);
    int rc = create_common(p);
    if (rc != FDD_OK) { destroy_plan(p); return rc; }
    *plan_out = p;
    return FDD_OK;
}

int fdd_plan_create_from_delays(fdd_plan** plan_out, int nchans, long long nsamps,
                                const double* delay_samples_host, int ndm)
{
    if (!plan_out) return FDD_ERR_INVALID_ARG;
    *plan_out = nullptr;
    if (nchans < 1 || nsamps < 2 || ndm < 1 || !delay_samples_host) return FDD_ERR_INVALID_ARG;
    for (size_t i = 0; i < (size_t)ndm * nchans; ++i)
        if (!isfinite(delay_samples_host[i])) return FDD_ERR_INVALID_ARG;
    fdd_plan* p = new (std::nothrow) fdd_plan();
    if (!p) return FDD_ERR_ALLOC;
    p->nchans = nchans; p->nsamps = nsamps; p->ndm = ndm; p->from_delays = true;
    p->delays.assign(delay_samples_host, delay_samples_host + (size_t)ndm * nchans);
    int rc = create_common(p);
    if (rc != FDD_OK) { destroy_plan(p); return rc; }
    *plan_out = p;
    return FDD_OK;
}

int fdd_plan_set_kdm(fdd_plan* p, double k_dm)
{
    if (check_plan(p) != FDD_OK || !(k_dm > 0) || !isfinite(k_dm)) return FDD_ERR_INVALID_ARG;
    if (p->from_delays) return FDD_ERR_UNSUPPORTED;
    DeviceGuard g(p->device);
    if (!g.ok || cudaDeviceSynchronize() != cudaSuccess) return FDD_ERR_CUDA;
    p->kdm = k_dm;
    build_delays(p);
    // the comparator's shift table follows the delays: drop it, it is rebuilt on next use
    if (p->tdd_shifts) {
        cudaFree(p->tdd_shifts); cudaFree(p->tdd_xt);
        p->scratch_bytes -= (size_t)p->nchans * p->ndm_pad * sizeof(int) + (size_t)p->nchans * p->tdd_tpitch;
        p->tdd_shifts = nullptr; p->tdd_xt = nullptr;
    }
    return build_tables(p);
}

int fdd_plan_set_decimation(fdd_plan* p, int log2_factor)
{
    if (check_plan(p) != FDD_OK || log2_factor < 0 || log2_factor > 30 || (p->nfft >> log2_factor) < 4)
        return FDD_ERR_INVALID_ARG;
    DeviceGuard g(p->device);
    if (!g.ok || cudaDeviceSynchronize() != cudaSuccess) return FDD_ERR_CUDA;
    // the TIME-mode resources depend on the output length: drop them, they are re-made by
    // fdd_plan_prepare or the next TIME execute
    drop_time_resources(p);
    p->log2_dec = log2_factor;
    p->nfft_out = p->nfft >> log2_factor;
    p->nbins_out = p->nfft_out / 2 + 1;
    p->nsamps_out = (p->nsamps + (1LL << log2_factor) - 1) >> log2_factor;
    return FDD_OK;
}

int fdd_plan_get_output_shape(const fdd_plan* p, long long* nsamps_out, long long* nbins_out)
{
    if (!p) return FDD_ERR_INVALID_ARG;
    if (nsamps_out) *nsamps_out = p->nsamps_out;
    if (nbins_out) *nbins_out = p->nbins_out;
    return FDD_OK;
}

int fdd_plan_set_kernel(fdd_plan* p, int kernel)
{
    if (check_plan(p) != FDD_OK) return FDD_ERR_INVALID_ARG;
    if (kernel < FDD_KERNEL_AUTO || kernel > FDD_KERNEL_TENSOR) return FDD_ERR_INVALID_ARG;
    if (kernel == FDD_KERNEL_TENSOR && !tensor_ok(p)) return FDD_ERR_UNSUPPORTED;
    if (kernel == FDD_KERNEL_MIXED && p->sym.nap == 0) return FDD_ERR_UNSUPPORTED;
    if (kernel == FDD_KERNEL_SYMMETRIC && !p->sym_ok) return FDD_ERR_UNSUPPORTED;
    if (kernel == FDD_KERNEL_SYMMETRIC2 && !p->sym_ok) return FDD_ERR_UNSUPPORTED;
    p->kernel_request = kernel;
    p->kernel = resolve_kernel(p, kernel);
    return FDD_OK;
}

int fdd_plan_set_inverse(fdd_plan* p, int which)
{
    if (check_plan(p) != FDD_OK ||
        (which != FDD_INVERSE_TWO_PASS && which != FDD_INVERSE_CUFFT && which != FDD_INVERSE_AUTO))
        return FDD_ERR_INVALID_ARG;
    DeviceGuard g(p->device);
    if (!g.ok || cudaDeviceSynchronize() != cudaSuccess) return FDD_ERR_CUDA;
    drop_time_resources(p);
    p->inverse_request = which;
    return FDD_OK;
}

int fdd_plan_get_inverse(const fdd_plan* p, int* which)
{
    if (!p || !which) return FDD_ERR_INVALID_ARG;
    *which = p->ifft_on ? FDD_INVERSE_TWO_PASS : FDD_INVERSE_CUFFT;
    return FDD_OK;
}

int fdd_plan_set_y_budget(fdd_plan* p, size_t bytes)
{
    if (check_plan(p) != FDD_OK) return FDD_ERR_INVALID_ARG;
    DeviceGuard g(p->device);
    if (!g.ok || cudaDeviceSynchronize() != cudaSuccess) return FDD_ERR_CUDA;
    drop_time_resources(p);
    p->y_budget = bytes;
    return FDD_OK;
}

int fdd_plan_prepare(fdd_plan* p, int mode)
{
    if (check_plan(p) != FDD_OK || (mode != FDD_MODE_TIME && mode != FDD_MODE_FOURIER))
        return FDD_ERR_INVALID_ARG;
    DeviceGuard g(p->device);
    if (!g.ok) return FDD_ERR_CUDA;
    int rc;
    int family = 0;
    if (mode == FDD_MODE_TIME && (rc = ensure_time_family(p, &family)) != FDD_OK) return rc;
    // the bin-recurrence tables, if any DM row can reach the generic kernel
    const bool generic_rows = p->kernel == FDD_KERNEL_GENERIC || p->kernel == FDD_KERNEL_MIXED ||
                              (mode == FDD_MODE_TIME && p->y_rows < p->ndm && p->y_rows % fdd::kSymT != 0);
    if (generic_rows && p->rec_pshift >= 0 && (rc = ensure_rec_tables(p, nullptr)) != FDD_OK) return rc;
    if ((rc = ensure_pad_table(p, nullptr)) != FDD_OK) return rc;
    // launch shapes of the shared-recurrence kernel for the chunks an execute will step through
    if (p->kernel == FDD_KERNEL_SYMMETRIC2) {
        const int step = mode == FDD_MODE_TIME ? p->y_rows : p->ndm;
        for (int j0 = 0; j0 < p->ndm && step % fdd::kSymT == 0; j0 += step) {
            const int rows = p->ndm - j0 < step ? p->ndm - j0 : step;
            if (!p->sym2_shapes.count(std::make_pair(j0, rows)))
                p->sym2_shapes.emplace(std::make_pair(j0, rows), fdd::sym2_shape(p->sym, j0, rows));
        }
    }
    if (cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); return FDD_ERR_CUDA; }
    return FDD_OK;
}

int fdd_execute(fdd_plan* p, const unsigned char* in_u8, void* out, int mode, void* cuda_stream)
{
    if (check_plan(p) != FDD_OK || !in_u8 || !out ||
        (mode != FDD_MODE_TIME && mode != FDD_MODE_FOURIER))
        return FDD_ERR_INVALID_ARG;
    DeviceGuard g(p->device);
    if (!g.ok) return FDD_ERR_CUDA;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    StageTimer tm(p, s);
    int rc = run_pre(p, in_u8, s, tm);
    if (rc != FDD_OK) return rc;
    return run_post(p, out, mode, s, tm, [](int, int) {}, 0, 0, [](int) {});
}

int fdd_rotate_sum_only(fdd_plan* p, void* out, int mode, void* cuda_stream)
{
    if (check_plan(p) != FDD_OK || !out || (mode != FDD_MODE_TIME && mode != FDD_MODE_FOURIER))
        return FDD_ERR_INVALID_ARG;
    DeviceGuard g(p->device);
    if (!g.ok) return FDD_ERR_CUDA;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    StageTimer tm(p, s);
    tm.begin(FDD_STAGE_ROTATE_SUM, 1);
    // FOURIER layout (pitch nbins) for either mode: `out` must hold ndm * nbins float2.
    int rc = launch_rotate_sum(p, 0, p->ndm, static_cast<float2*>(out), p->nbins_out, mode, s);
    tm.end();
    return rc;
}

int fdd_execute_host(fdd_plan* p, const unsigned char* in_host, void* out_host, int mode,
                     void* cuda_stream)
{
    if (check_plan(p) != FDD_OK || !in_host || !out_host ||
        (mode != FDD_MODE_TIME && mode != FDD_MODE_FOURIER))
        return FDD_ERR_INVALID_ARG;
    DeviceGuard g(p->device);
    if (!g.ok) return FDD_ERR_CUDA;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t in_bytes = (size_t)p->nsamps * p->nchans;
    const size_t row_bytes = mode == FDD_MODE_TIME ? (size_t)p->nsamps_out * sizeof(float)
                                                   : (size_t)p->nbins_out * sizeof(float2);
    // The device side of the output is a ring of kHostRingChunks chunks (Algorithm 1's output
    // buffers): results may be larger than HBM, only the host array holds them all.
    int rc;
    int family = 0;
    if (mode == FDD_MODE_TIME && (rc = ensure_time_family(p, &family)) != FDD_OK) return rc;
    // chunk = what run_post will step by: kHostChunkRows, or the whole Y scratch if that is smaller
    const int chunk = (mode == FDD_MODE_TIME && p->y_rows < kHostChunkRows) ? p->y_rows : kHostChunkRows;
    const int ring_rows = kHostRingChunks * chunk;
    const size_t out_bytes = row_bytes * (size_t)(p->ndm < ring_rows ? p->ndm : ring_rows);
    if (!p->stage_in && (rc = dev_alloc(p, &p->stage_in, in_bytes)) != FDD_OK) return rc;
    if (p->stage_out_bytes < out_bytes) {
        if (p->stage_out) { cudaFree(p->stage_out); p->scratch_bytes -= p->stage_out_bytes; p->stage_out = nullptr; }
        p->stage_out_bytes = 0;
        if ((rc = dev_alloc(p, reinterpret_cast<unsigned char**>(&p->stage_out), out_bytes)) != FDD_OK)
            return rc;
        p->stage_out_bytes = out_bytes;
    }
    if (!p->copy_stream &&
        cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking) != cudaSuccess)
        return FDD_ERR_CUDA;
    // Algorithm 1 lines 9-17: the input goes up in time blocks on the copy stream and every block is
    // unpacked as soon as it has landed (a2 is local in time; only the R2C needs whole rows)
    StageTimer tm(p, s);
    {
        constexpr int kInBlocks = 8;
        while (p->in_events.size() < (size_t)kInBlocks) {
            cudaEvent_t e;
            if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return FDD_ERR_CUDA; }
            p->in_events.push_back(e);
        }
        const long long data_tiles = (p->nsamps + fdd::kUnpackTile - 1) / fdd::kUnpackTile;
        const long long all_tiles = (p->nfft + fdd::kUnpackTile - 1) / fdd::kUnpackTile;
        // (the copy stream must not run ahead of work still queued on s from an earlier call)
        cudaEvent_t start = p->in_events[0];
        if (cudaEventRecord(start, s) != cudaSuccess || cudaStreamWaitEvent(p->copy_stream, start, 0) != cudaSuccess)
            return FDD_ERR_CUDA;
        tm.begin(FDD_STAGE_UNPACK, kInBlocks);
        for (int b = 0; b < kInBlocks; ++b) {
            const long long tl = data_tiles * b / kInBlocks, th = b + 1 < kInBlocks ? data_tiles * (b + 1) / kInBlocks : all_tiles;
            const long long t_lo = tl * fdd::kUnpackTile;
            long long t_hi = th * fdd::kUnpackTile;
            if (t_hi > p->nsamps) t_hi = p->nsamps;
            if (t_hi > t_lo &&
                cudaMemcpyAsync(p->stage_in + (size_t)t_lo * p->nchans, in_host + (size_t)t_lo * p->nchans,
                                (size_t)(t_hi - t_lo) * p->nchans, cudaMemcpyHostToDevice, p->copy_stream) != cudaSuccess)
                return FDD_ERR_CUDA;
            if (cudaEventRecord(p->in_events[b], p->copy_stream) != cudaSuccess ||
                cudaStreamWaitEvent(s, p->in_events[b], 0) != cudaSuccess)
                return FDD_ERR_CUDA;
            if ((rc = launch_unpack(p, p->stage_in, s, tl, th - tl)) != FDD_OK) return rc;
        }
        tm.end();
    }
    rc = run_pre(p, p->stage_in, s, tm, true);
    if (rc != FDD_OK) return rc;
    // two events per chunk: [2i] results ready (on s), [2i+1] copied back (on copy_stream)
    const int nchunks = (p->ndm + chunk - 1) / chunk;
    while (p->chunk_events.size() < (size_t)2 * nchunks) {
        cudaEvent_t e;
        if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            return FDD_ERR_CUDA;
        }
        p->chunk_events.push_back(e);
    }
    bool copy_fail = false;
    // a ring slot is rewritten only after the chunk that used it last has been copied back
    auto chunk_begin = [&](int j0) {
        const int i = j0 / chunk;
        if (i >= kHostRingChunks &&
            cudaStreamWaitEvent(s, p->chunk_events[2 * (i - kHostRingChunks) + 1], 0) != cudaSuccess)
            copy_fail = true;
    };
    // Algorithm 1 lines 19-22: copy each finished DM chunk back while later chunks still compute.
    auto chunk_done = [&](int j0, int rows) {
        const int i = j0 / chunk;
        cudaEvent_t ready = p->chunk_events[2 * i], copied = p->chunk_events[2 * i + 1];
        if (cudaEventRecord(ready, s) != cudaSuccess ||
            cudaStreamWaitEvent(p->copy_stream, ready, 0) != cudaSuccess ||
            cudaMemcpyAsync(static_cast<char*>(out_host) + (size_t)j0 * row_bytes,
                            static_cast<char*>(p->stage_out) + (size_t)(j0 % ring_rows) * row_bytes,
                            (size_t)rows * row_bytes, cudaMemcpyDeviceToHost,
                            p->copy_stream) != cudaSuccess ||
            cudaEventRecord(copied, p->copy_stream) != cudaSuccess)
            copy_fail = true;
    };
    // DM chunks of kHostChunkRows rows: the copy back of chunk i overlaps the compute of chunk i+1
    rc = run_post(p, p->stage_out, mode, s, tm, chunk_done, chunk, ring_rows, chunk_begin);
    if (rc != FDD_OK) return rc;
    if (copy_fail) { cudaGetLastError(); return FDD_ERR_CUDA; }
    if (cudaStreamSynchronize(p->copy_stream) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess) {
        cudaGetLastError();
        return FDD_ERR_CUDA;
    }
    return FDD_OK;
}

int fdd_tdd_execute(fdd_plan* p, const unsigned char* in_u8, float* out, void* cuda_stream)
{
    if (check_plan(p) != FDD_OK || !in_u8 || !out) return FDD_ERR_INVALID_ARG;
    DeviceGuard g(p->device);
    if (!g.ok) return FDD_ERR_CUDA;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    int rc;
    if (!p->tdd_shifts) {
        // Eq. 2: shifts rounded to the nearest sample, reduced mod nsamps (the result is circular)
        std::vector<int> sh((size_t)p->nchans * p->ndm_pad, 0);
        long long smax = 0;
        for (int j = 0; j < p->ndm; ++j)
            for (int c = 0; c < p->nchans; ++c) {
                long long v = (long long)floor(p->delays[(size_t)j * p->nchans + c] + 0.5) % p->nsamps;
                if (v < 0) v += p->nsamps;
                sh[(size_t)c * p->ndm_pad + j] = (int)v;
                if (v > smax) smax = v;
            }
        if (p->nsamps > 2147483647LL - 256) return FDD_ERR_UNSUPPORTED;
        p->tdd_tpitch = round_up(p->nsamps + smax + 128, 64);
        if ((rc = dev_alloc(p, &p->tdd_shifts, sh.size())) != FDD_OK) return rc;
        if ((rc = dev_alloc(p, &p->tdd_xt, (size_t)p->nchans * p->tdd_tpitch)) != FDD_OK) return rc;
        if (cudaMemcpy(p->tdd_shifts, sh.data(), sh.size() * sizeof(int), cudaMemcpyHostToDevice) !=
            cudaSuccess) {
            cudaGetLastError();
            return FDD_ERR_CUDA;
        }
    }
    StageTimer tm(p, s);
    tm.begin(FDD_STAGE_TDD_TRANSPOSE, 1);
    dim3 tgrid((unsigned)(p->tdd_tpitch / 64), (unsigned)((p->nchans + 63) / 64));
    fdd::k_tdd_transpose<<<tgrid, 256, 0, s>>>(in_u8, p->tdd_xt, p->nchans, p->nsamps, p->tdd_tpitch);
    tm.end();
    if (cudaGetLastError() != cudaSuccess) return FDD_ERR_CUDA;
    const int ntiles_dm = (p->ndm + fdd::kTddDms - 1) / fdd::kTddDms;
    const long long ntb = (p->nsamps + fdd::kTddTile - 1) / fdd::kTddTile;
    if ((long long)ntiles_dm * ntb > 2147483647LL) return FDD_ERR_UNSUPPORTED;
    tm.begin(FDD_STAGE_TDD_SHIFT_ADD, 1);
    fdd::k_tdd_shift_add<<<(unsigned)(ntiles_dm * ntb), fdd::kTddWarps * 32, 0, s>>>(
        p->tdd_xt, p->tdd_tpitch, p->tdd_shifts, p->ndm_pad, p->nchans, p->nsamps, p->ndm, ntiles_dm,
        out);
    tm.end();
    return cudaGetLastError() == cudaSuccess ? FDD_OK : FDD_ERR_CUDA;
}

int fdd_execute_beams(fdd_plan* p, const unsigned char* in_u8, void* out, int nbeams, int mode,
                      void* cuda_stream)
{
    if (check_plan(p) != FDD_OK || !in_u8 || !out || nbeams < 1 ||
        (mode != FDD_MODE_TIME && mode != FDD_MODE_FOURIER))
        return FDD_ERR_INVALID_ARG;
    DeviceGuard g(p->device);
    if (!g.ok) return FDD_ERR_CUDA;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t in_beam = (size_t)p->nsamps * p->nchans;
    const size_t out_beam = mode == FDD_MODE_TIME ? (size_t)p->ndm * p->nsamps_out * sizeof(float)
                                                  : (size_t)p->ndm * p->nbins_out * sizeof(float2);
    // beams per tensor-core launch: the 64 tile rows of its Z operand are shared out between them
    int group = 1;
    const bool tensor = tensor_ok(p) && (p->kernel_request == FDD_KERNEL_AUTO || p->kernel_request == FDD_KERNEL_TENSOR);
    if (tensor && nbeams > 1) group = p->ndm <= 1024 ? 4 : (p->ndm <= 2048 ? 2 : 1);
    int rc;
    int family = 0;
    if (group > 1 && mode == FDD_MODE_TIME) {
        if ((rc = ensure_time_resources(p, 0)) != FDD_OK) return rc;
        if (p->y_rows != p->ndm) group = 1;               // (Y is chunked: one beam at a time)
    }
    StageTimer tm(p, s);
    if (group == 1) {
        // no sharing possible (more than 2048 trial DMs, or not a uniform DM grid): beam after beam
        for (int b = 0; b < nbeams; ++b) {
            if ((rc = run_pre(p, in_u8 + (size_t)b * in_beam, s, tm)) != FDD_OK) return rc;
            rc = run_post(p, static_cast<char*>(out) + (size_t)b * out_beam, mode, s, tm, [](int, int) {}, 0, 0,
                          [](int) {});
            if (rc != FDD_OK) return rc;
        }
        return FDD_OK;
    }
    if (p->beam_group < group) {
        if (cudaDeviceSynchronize() != cudaSuccess) return FDD_ERR_CUDA;
        if (p->beam_X) { cudaFree(p->beam_X); p->scratch_bytes -= (size_t)p->beam_group * p->nchans * p->xpitch * sizeof(float2); p->beam_X = nullptr; }
        if (p->beam_Y) { cudaFree(p->beam_Y); p->scratch_bytes -= (size_t)p->beam_group * p->ndm * p->ypitch * sizeof(float2); p->beam_Y = nullptr; }
        p->beam_group = 0;
        if ((rc = dev_alloc(p, &p->beam_X, (size_t)group * p->nchans * p->xpitch)) != FDD_OK) return rc;
        p->beam_group = group;
    }
    if (mode == FDD_MODE_TIME && !p->beam_Y &&
        (rc = dev_alloc(p, &p->beam_Y, (size_t)p->beam_group * p->ndm * p->ypitch)) != FDD_OK)
        return rc;
    const float scale = mode == FDD_MODE_TIME ? (float)(1.0 / (double)p->nfft) : 1.0f;
    const double dc_raw = p->padded ? 0.0 : (double)p->offset * (double)p->nchans * (double)p->nsamps;
    if (mode == FDD_MODE_TIME && (rc = ensure_time_family(p, &family)) != FDD_OK) return rc;
    const float dc_add = mode == FDD_MODE_TIME ? (p->ifft_on ? 0.f : (float)(dc_raw / (double)p->nfft)) : (float)dc_raw;
    int e = 0;
    frexp((p->padded ? 256.0 : 128.0) * (double)p->nsamps, &e);
    const float xscale = (float)ldexp(1.0, 15 - e);
    const long long xstride = (long long)p->nchans * p->xpitch;
    for (int b0 = 0; b0 < nbeams; b0 += group) {
        const int gb = nbeams - b0 < group ? nbeams - b0 : group;
        const int glaunch = gb == 3 ? 0 : gb;
        for (int b = 0; b < gb; ++b) {
            // a2 + a3 of beam b0 + b into its slot of beam_X
            tm.begin(FDD_STAGE_UNPACK, 1);
            rc = launch_unpack(p, in_u8 + (size_t)(b0 + b) * in_beam, s, 0, -1, p->beam_X + (long long)b * xstride);
            tm.end();
            if (rc != FDD_OK) return rc;
            tm.begin(FDD_STAGE_R2C, 1);
            if (cufftSetStream(p->r2c, s) != CUFFT_SUCCESS) return FDD_ERR_CUFFT;
            if (cufftExecR2C(p->r2c,
                             p->r2c_inplace ? reinterpret_cast<float*>(p->beam_X + (long long)b * xstride) : p->xreal,
                             p->beam_X + (long long)b * xstride) != CUFFT_SUCCESS)
                return FDD_ERR_CUFFT;
            rc = launch_pad_add_rect(p, p->beam_X + (long long)b * xstride, s);
            tm.end();
            if (rc != FDD_OK) return rc;
        }
        // a4 for the whole group: one launch, the pair phasors are made once for all its beams
        // (the kernel shares its operand rows among 1, 2 or 4 beams: a group of 3 runs as 2 + 1)
        float2* dst = mode == FDD_MODE_TIME ? p->beam_Y
                                            : static_cast<float2*>(out) + (size_t)b0 * p->ndm * p->nbins_out;
        const long long opitch = mode == FDD_MODE_TIME ? p->ypitch : p->nbins_out;
        const long long ostride = (long long)p->ndm * opitch;
        tm.begin(FDD_STAGE_ROTATE_SUM, 1);
        if (glaunch == gb) {
            rc = fdd::tc_launch(p->sym, p->nfft, p->beam_X, p->xpitch, p->nchans, p->nbins_out, p->ndm, 0, p->ndm,
                                dst, opitch, scale, mode == FDD_MODE_TIME ? 1 : 0, dc_add, xscale, p->num_sms, s,
                                glaunch, xstride, ostride);
        } else {
            rc = fdd::tc_launch(p->sym, p->nfft, p->beam_X, p->xpitch, p->nchans, p->nbins_out, p->ndm, 0, p->ndm,
                                dst, opitch, scale, mode == FDD_MODE_TIME ? 1 : 0, dc_add, xscale, p->num_sms, s,
                                2, xstride, ostride);
            if (rc == 0)
                rc = fdd::tc_launch(p->sym, p->nfft, p->beam_X + 2 * xstride, p->xpitch, p->nchans, p->nbins_out,
                                    p->ndm, 0, p->ndm, dst + 2 * ostride, opitch, scale,
                                    mode == FDD_MODE_TIME ? 1 : 0, dc_add, xscale, p->num_sms, s, 1, 0, 0);
        }
        for (int b = 0; b < gb && rc == 0; ++b)
            rc = launch_pad_add_table(p, 0, p->ndm, dst + (long long)b * ostride, opitch, mode, s);
        tm.end();
        if (rc != 0) return rc == -5 ? FDD_ERR_UNSUPPORTED : (rc < 0 && rc > -5 ? rc : FDD_ERR_CUDA);
        if (mode == FDD_MODE_TIME) {
            for (int b = 0; b < gb; ++b) {
                int nl = 0;
                tm.begin(FDD_STAGE_C2R, 0);
                rc = launch_c2r_rows(p, 0, p->ndm, p->beam_Y + (long long)b * ostride,
                                     static_cast<float*>(out) + (size_t)(b0 + b) * p->ndm * p->nsamps_out, s, &nl);
                tm.end();
                p->launches[FDD_STAGE_C2R] += nl;
                if (rc != FDD_OK) return rc;
            }
        }
    }
    return FDD_OK;
}

int fdd_tc_selftest(const void* a_f16_dev, const void* b_f16_dev, float* d_dev, void* cuda_stream)
{
    if (!a_f16_dev || !b_f16_dev || !d_dev) return FDD_ERR_INVALID_ARG;
    const int smem = 1024 + fdd::kTcZBytes + fdd::kTcEBytes + 64;
    if (cudaFuncSetAttribute(fdd::k_tc_selftest, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) {
        cudaGetLastError();
        return FDD_ERR_CUDA;
    }
    fdd::k_tc_selftest<<<1, 128, smem, static_cast<cudaStream_t>(cuda_stream)>>>(
        static_cast<const __half*>(a_f16_dev), static_cast<const __half*>(b_f16_dev), d_dev);
    return cudaGetLastError() == cudaSuccess ? FDD_OK : FDD_ERR_CUDA;
}

int fdd_plan_destroy(fdd_plan* p)
{
    destroy_plan(p);
    return FDD_OK;
}

int fdd_plan_get_info(const fdd_plan* p, long long* nfft, long long* nbins, long long* valid_len,
                      double* max_delay_samples, size_t* scratch_bytes, int* kernel)
{
    if (!p) return FDD_ERR_INVALID_ARG;
    if (nfft) *nfft = p->nfft;
    if (nbins) *nbins = p->nbins;
    if (valid_len) *valid_len = p->valid_len;
    if (max_delay_samples) *max_delay_samples = p->max_delay;
    if (scratch_bytes) *scratch_bytes = p->scratch_bytes;
    if (kernel) *kernel = p->kernel;
    return FDD_OK;
}

int fdd_plan_get_delays(const fdd_plan* p, double* delay_samples_host)
{
    if (!p || !delay_samples_host) return FDD_ERR_INVALID_ARG;
    memcpy(delay_samples_host, p->delays.data(), p->delays.size() * sizeof(double));
    return FDD_OK;
}

int fdd_plan_set_profiling(fdd_plan* p, int enable)
{
    if (!p) return FDD_ERR_INVALID_ARG;
    p->profiling = enable != 0;
    reset_profile(p);
    return FDD_OK;
}

int fdd_plan_get_stage_ms(fdd_plan* p, float* ms_host, int* launches_host)
{
    if (!p || !ms_host) return FDD_ERR_INVALID_ARG;
    DeviceGuard g(p->device);
    for (int i = 0; i < FDD_NUM_STAGES; ++i) ms_host[i] = 0.f;
    for (size_t i = 0; i < p->events_used; ++i) {
        StageEvent& e = p->events[i];
        if (cudaEventSynchronize(e.end) != cudaSuccess) { cudaGetLastError(); return FDD_ERR_CUDA; }
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, e.beg, e.end) != cudaSuccess) { cudaGetLastError(); return FDD_ERR_CUDA; }
        ms_host[e.stage] += ms;
    }
    if (launches_host)
        for (int i = 0; i < FDD_NUM_STAGES; ++i) launches_host[i] = p->launches[i];
    return FDD_OK;
}

int fdd_plan_get_spectrum(const fdd_plan* p, void** x_dev, long long* pitch_elems,
                          double* dc_removed)
{
    if (!p || !x_dev || !pitch_elems) return FDD_ERR_INVALID_ARG;
    *x_dev = p->X;
    *pitch_elems = p->xpitch;
    if (dc_removed) *dc_removed = (double)p->offset * (double)p->nsamps;
    return FDD_OK;
}

int fdd_plan_get_padding(const fdd_plan* p, long long* exact_bins)
{
    if (!p || !exact_bins) return FDD_ERR_INVALID_ARG;
    *exact_bins = p->padded ? p->pad_k : 0;
    return FDD_OK;
}

int fdd_measure_fp32_peak(int packed, int iters, double* tflops_host, float* ms_host)
{
    if (iters < 1 || !tflops_host) return FDD_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return FDD_ERR_CUDA;
    }
    float* sink = nullptr;
    cudaEvent_t a = nullptr, b = nullptr;
    int rc = FDD_ERR_CUDA;
    const int blocks = sms * 8, threads = 256;
    float ms = 0.f;
    if (cudaMalloc(&sink, sizeof(float)) != cudaSuccess) { cudaGetLastError(); return FDD_ERR_ALLOC; }
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) goto done;
    for (int rep = 0; rep < 2; ++rep) {          // first launch warms up
        cudaEventRecord(a, 0);
        if (packed) fdd::k_fp32_peak<true><<<blocks, threads>>>(sink, iters, 0.999f, 1e-3f);
        else fdd::k_fp32_peak<false><<<blocks, threads>>>(sink, iters, 0.999f, 1e-3f);
        cudaEventRecord(b, 0);
        if (cudaEventSynchronize(b) != cudaSuccess) goto done;
        cudaEventElapsedTime(&ms, a, b);
    }
    if (cudaGetLastError() != cudaSuccess) goto done;
    // per thread per iteration: 4 unrolls * 8 chains * 2 lanes FMA = 64 FMA = 128 flop
    *tflops_host = (double)blocks * threads * (double)iters * 128.0 / (ms * 1e-3) * 1e-12;
    if (ms_host) *ms_host = ms;
    rc = FDD_OK;
done:
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    cudaFree(sink);
    cudaGetLastError();
    return rc;
}

const char* fdd_error_string(int status)
{
    switch (status) {
        case FDD_OK: return "ok";
        case FDD_ERR_INVALID_ARG: return "invalid argument";
        case FDD_ERR_ALLOC: return "out of memory";
        case FDD_ERR_CUDA: return "CUDA error";
        case FDD_ERR_CUFFT: return "cuFFT error";
        case FDD_ERR_UNSUPPORTED: return "unsupported";
        case FDD_ERR_TOO_LARGE: return "problem larger than the static scratch (FDD_STATIC_MAX_PHASES)";
        default: return "unknown status";
    }
}

}  // extern "C"
