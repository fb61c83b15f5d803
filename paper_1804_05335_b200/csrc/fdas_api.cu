// C ABI of the FDAS library (see include/fdas.h).  Host logic only: argument checks, plan
// geometry, device allocations, kernel dispatch.  Every step of the path runs in the kernels
// of fdas_templates.cuh / fdas_kernel.cuh; there is no CPU fallback.
#include "../../include/fdas.h"
#include "fdas_templates.cuh"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

using namespace fdas;

static std::atomic<long long> g_launches{0};

struct fdas_plan {
    fdas_info info;
    int device;
    bool ready;
    int nbanks;          // 2 with two-bin Fourier interpolation (bank 1: half-bin templates)
    double2 *d_taps;     // K x (2m+1)
    float2 *d_hperm;     // npairs x L (kernel register order)
    float2 *d_wtab;      // L (seglen 8192: the 4096 table)
    float2 *d_wtab2;     // seglen 8192 only: 8192 entries
    float2 *d_stage_in;  // fdas_execute_host staging (lazy)
    float *d_stage_out;
    fdas_candidate *d_stage_cands;   // fdas_execute_threshold_host staging (lazy, grows with capacity)
    int64_t stage_cands_cap;
    unsigned long long *d_stage_count;
    void (*kernel)(const KernelParams);
    void (*kernel_thr)(const KernelParams);   // MODE 1: threshold search instead of the plane store
    char err[256];
};

#define FDAS_CUDA(plan, call)                                                                  \
    do {                                                                                       \
        cudaError_t e__ = (call);                                                              \
        if (e__ != cudaSuccess) {                                                              \
            if (plan)                                                                          \
                snprintf((plan)->err, sizeof((plan)->err), "%s: %s", #call,                    \
                         cudaGetErrorString(e__));                                             \
            return FDAS_ERR_CUDA;                                                              \
        }                                                                                      \
    } while (0)

namespace {

// Text of the last failure inside fdas_plan_create (the plan is gone by then): fdas_last_error(NULL).
thread_local char g_create_err[256] = "";

// Plans are bound to the device that was current at fdas_plan_create: every entry point that touches
// plan-owned device memory refuses to run with another device current (FDAS_ERR_INVALID_ARG).
bool on_plan_device(fdas_plan *p)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    if (dev != p->device) {
        snprintf(p->err, sizeof(p->err), "plan was created on device %d, current device is %d", p->device, dev);
        return false;
    }
    return true;
}

typedef void (*kernel_fn)(const KernelParams);

template <int L, int MINB>
kernel_fn pick_kernel(int ib, int mode)
{
    if (ib == 2) return mode ? (kernel_fn)fdas_fused_kernel<L, false, MINB, 1, 2> : (kernel_fn)fdas_fused_kernel<L, false, MINB, 0, 2>;
    if (mode) return ib ? (kernel_fn)fdas_fused_kernel<L, true, MINB, 1> : (kernel_fn)fdas_fused_kernel<L, false, MINB, 1>;
    return ib ? (kernel_fn)fdas_fused_kernel<L, true, MINB> : (kernel_fn)fdas_fused_kernel<L, false, MINB>;
}

// L = 4096: second-generation kernel (shuffle exchange, fdas_kernel2.cuh).
template <int L, int MINB>
kernel_fn pick_kernel2(int ib, int mode)
{
    if (ib == 2) return mode ? (kernel_fn)fdas_fused_kernel2<L, false, MINB, 1, 2> : (kernel_fn)fdas_fused_kernel2<L, false, MINB, 0, 2>;
    if (mode) return ib ? (kernel_fn)fdas_fused_kernel2<L, true, MINB, 1> : (kernel_fn)fdas_fused_kernel2<L, false, MINB, 1>;
    return ib ? (kernel_fn)fdas_fused_kernel2<L, true, MINB> : (kernel_fn)fdas_fused_kernel2<L, false, MINB>;
}

// L = 2048: third-generation kernel (X^ and twiddles in tensor memory, three CTAs per SM, fdas_kernel3.cuh);
// L = 4096 interbinned: the same kernel with X^ and twiddles in registers (one CTA per SM).
template <int L, int MINB>
kernel_fn pick_kernel3(int ib, int mode)
{
    if (ib == 2) return mode ? (kernel_fn)fdas_fused_kernel3<L, false, MINB, 1, 2> : (kernel_fn)fdas_fused_kernel3<L, false, MINB, 0, 2>;
    if (mode) return ib ? (kernel_fn)fdas_fused_kernel3<L, true, MINB, 1> : (kernel_fn)fdas_fused_kernel3<L, false, MINB, 1>;
    return ib ? (kernel_fn)fdas_fused_kernel3<L, true, MINB> : (kernel_fn)fdas_fused_kernel3<L, false, MINB>;
}

constexpr int K3_CTAS_PER_SM_2048 = 3;   // fdas_kernel3.cuh at L = 2048: <= 168 registers, 72 KB, 128 tensor-memory columns

// mode 0: plane store (fdas_execute); mode 1: threshold search (fdas_execute_threshold)
// ib: 0 none, 1 interbinning (eq. 4), 2 two-bin Fourier interpolation (second template bank)
kernel_fn select_kernel(int L, int ib, int mode = 0)
{
    // debug aid (include/fdas.h, fdas_plan_create): the 8192 plane kernels with a CTA barrier in front of every E1 store
    if (L == 8192 && mode == 0) {
        const char *dbg = std::getenv("FDAS_DEBUG_E1_SYNC");
        if (dbg && dbg[0] == '1') {
            if (ib == 2) return (kernel_fn)fdas_fused_kernel_8k<1, 0, false, 2, true>;
            return ib ? (kernel_fn)fdas_fused_kernel_8k<1, 0, true, 1, true> : (kernel_fn)fdas_fused_kernel_8k<1, 0, false, 1, true>;
        }
    }
    switch (L) {
    case 1024: return pick_kernel<1024, 4>(ib, mode);
    case 2048: return pick_kernel3<2048, K3_CTAS_PER_SM_2048>(ib, mode);
    case 4096:                                                            // measured per half-bin mode
        return ib == 1 ? pick_kernel3<4096, 1>(ib, mode) : pick_kernel2<4096, 1>(ib, mode);
    case 8192:                                                            // 2 x 4096 (fdas_kernel8k.cuh)
        if (ib == 2) return mode ? (kernel_fn)fdas_fused_kernel_8k<1, 1, false, 2> : (kernel_fn)fdas_fused_kernel_8k<1, 0, false, 2>;
        if (ib) return mode ? (kernel_fn)fdas_fused_kernel_8k<1, 1, true> : (kernel_fn)fdas_fused_kernel_8k<1, 0, true>;
        return mode ? (kernel_fn)fdas_fused_kernel_8k<1, 1> : (kernel_fn)fdas_fused_kernel_8k<1>;
    default: return nullptr;
    }
}

int smem_bytes_for(int L, bool ib)
{
    switch (L) {
    case 1024: return Geo<1024>::smem_bytes(ib);
    case 2048: return Geo3<2048>::smem_bytes(ib);
    case 4096: return ib ? Geo3<4096>::smem_bytes(true) : Geo2<4096>::smem_bytes(false);
    case 8192: return Geo8k::smem_bytes();
    default: return 0;
    }
}

// Tensor-memory columns one CTA of the selected kernel allocates (0: none).  L = 4096 runs without parking.
int tmem_cols_for(int L)
{
    switch (L) {
    case 2048: return Geo3<2048>::TM_COLS;
    case 8192: return Geo8k::TM_COLS;
    default: return 0;
    }
}

// CTAs of one kernel an SM can hold at once, from the device's limits: registers (allocated per warp in units of 8
// per thread), shared memory (dynamic + static + the per-CTA reserve), the 512 tensor-memory columns, threads and
// CTA slots.  cudaOccupancyMaxActiveBlocksPerMultiprocessor cannot be asked: it answers 1 for every kernel that
// allocates tensor memory.
int resident_ctas(const cudaDeviceProp &prop, const cudaFuncAttributes &fa, int threads, int smem_dyn, int tm_cols)
{
    const long long regs_cta = (long long)((fa.numRegs + 7) / 8 * 8) * ((threads + 31) / 32 * 32);
    const long long smem_cta = (long long)smem_dyn + (long long)fa.sharedSizeBytes + (long long)prop.reservedSharedMemPerBlock;
    long long n = prop.maxBlocksPerMultiProcessor;
    if (regs_cta > 0 && prop.regsPerMultiprocessor / regs_cta < n) n = prop.regsPerMultiprocessor / regs_cta;
    if (smem_cta > 0 && (long long)prop.sharedMemPerMultiprocessor / smem_cta < n) n = (long long)prop.sharedMemPerMultiprocessor / smem_cta;
    if (tm_cols > 0 && 512 / tm_cols < n) n = 512 / tm_cols;
    if (prop.maxThreadsPerMultiProcessor / threads < n) n = prop.maxThreadsPerMultiProcessor / threads;
    return (int)n;
}

void freq_to_reg_any(int L, int f, int &tid, int &i)
{
    switch (L) {
    case 1024: freq_to_reg<1024>(f, tid, i); break;
    case 2048: freq_to_reg3<2048>(f, tid, i); break;
    default: freq_to_reg<4096>(f & 4095, tid, i); break;   // 8192: slot of f mod 4096 in half f / 4096
    }
}

} // namespace

extern "C" {

const char *fdas_status_string(fdas_status s)
{
    switch (s) {
    case FDAS_OK: return "FDAS_OK";
    case FDAS_ERR_INVALID_ARG: return "FDAS_ERR_INVALID_ARG";
    case FDAS_ERR_UNSUPPORTED: return "FDAS_ERR_UNSUPPORTED";
    case FDAS_ERR_NOT_READY: return "FDAS_ERR_NOT_READY";
    case FDAS_ERR_ALIGNMENT: return "FDAS_ERR_ALIGNMENT";
    case FDAS_ERR_CUDA: return "FDAS_ERR_CUDA";
    case FDAS_ERR_NOMEM: return "FDAS_ERR_NOMEM";
    }
    return "FDAS_ERR_UNKNOWN";
}

const char *fdas_last_error(const fdas_plan *plan) { return plan ? plan->err : g_create_err; }

int64_t fdas_launch_count(void) { return g_launches.load(); }

fdas_status fdas_plan_create(fdas_plan **out, int64_t nbins, double zmax, double dz, int32_t seglen,
                             int32_t interbin)
{
    if (!out) return FDAS_ERR_INVALID_ARG;
    *out = nullptr;
    if (nbins <= 0 || !(zmax >= 0.0) || !(dz > 0.0) || !std::isfinite(zmax) || !std::isfinite(dz))
        return FDAS_ERR_INVALID_ARG;
    const double nh = zmax / dz;
    const double nhr = std::floor(nh + 0.5);
    if (std::fabs(nh - nhr) > 1e-9 * std::fmax(1.0, nh) || nhr > 1e6) return FDAS_ERR_INVALID_ARG;
    if (interbin < 0 || interbin > 2) return FDAS_ERR_INVALID_ARG;
    if (seglen != 1024 && seglen != 2048 && seglen != 4096 && seglen != 8192)
        return FDAS_ERR_UNSUPPORTED;

    const int K = 2 * (int)nhr + 1;
    const int m = (int)std::ceil(zmax * 0.5 - 1e-12) + 16;
    const int ov = ((m + (interbin ? 1 : 0)) + 31) / 32 * 32; // >= m (+1 for the interbin neighbour), 128B-aligned
    const int B = seglen - 2 * ov;
    if (B < 32) return FDAS_ERR_UNSUPPORTED;
    g_create_err[0] = 0;
    // 32-bit index arithmetic in the template kernels: K * (2m+1) taps and npairs * L spectrum slots per bank
    if ((double)K * (2.0 * m + 1.0) > 2.0e9 || ((double)K + 1.0) * 0.5 * seglen > 2.0e9) {
        snprintf(g_create_err, sizeof(g_create_err), "template bank too large: K = %d, half-width %d", K, m);
        return FDAS_ERR_UNSUPPORTED;
    }
    kernel_fn kern = select_kernel(seglen, interbin);
    if (!kern) return FDAS_ERR_UNSUPPORTED;

    fdas_plan *p = new (std::nothrow) fdas_plan();
    if (!p) return FDAS_ERR_NOMEM;
    std::memset(p, 0, sizeof(*p));
    p->kernel = kern;
    p->kernel_thr = select_kernel(seglen, interbin, 1);
    p->nbanks = interbin == 2 ? 2 : 1;
    fdas_info &I = p->info;
    I.nbins = nbins;
    I.ncols = interbin ? 2 * nbins : nbins;
    I.row_stride = I.ncols;
    I.nseg = (nbins + B - 1) / B;
    I.plane_bytes = (int64_t)K * I.ncols * 4;
    I.zmax = zmax;
    I.dz = dz;
    I.ntemplates = K;
    I.seglen = seglen;
    I.halfwidth = m;
    I.overlap = ov;
    I.useful = B;
    I.interbin = interbin;
    I.npairs = (K + 1) / 2;
    I.threads = seglen == 8192 ? 256 : seglen / 16;
    I.smem_bytes = smem_bytes_for(seglen, interbin == 1);

    fdas_status st = FDAS_OK;
    do {
        cudaError_t e = cudaSuccess;
#define FDAS_CREATE_FAIL(code)                                                                     \
    {                                                                                              \
        st = code;                                                                                 \
        snprintf(g_create_err, sizeof(g_create_err), "fdas_plan_create: %s", cudaGetErrorString(e)); \
        break;                                                                                     \
    }
        if ((e = cudaGetDevice(&p->device)) != cudaSuccess) FDAS_CREATE_FAIL(FDAS_ERR_CUDA)
        cudaDeviceProp prop;
        if ((e = cudaGetDeviceProperties(&prop, p->device)) != cudaSuccess) FDAS_CREATE_FAIL(FDAS_ERR_CUDA)
        I.sm_count = prop.multiProcessorCount;
        if ((e = cudaFuncSetAttribute((const void *)kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      I.smem_bytes)) != cudaSuccess) FDAS_CREATE_FAIL(FDAS_ERR_CUDA)
        if ((e = cudaFuncSetAttribute((const void *)p->kernel_thr, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      I.smem_bytes)) != cudaSuccess) FDAS_CREATE_FAIL(FDAS_ERR_CUDA)
        // three 72 KB CTAs per SM (L = 2048) only fit with the largest shared-memory carve-out of the unified L1; the
        // other kernels keep the driver's choice, which leaves them more L1 for the `H` loads (measured on L = 4096:
        // 1.857 ms with the default carve-out, 1.935 ms with the maximum)
        if (seglen == 2048) {
            if ((e = cudaFuncSetAttribute((const void *)kern, cudaFuncAttributePreferredSharedMemoryCarveout,
                                          cudaSharedmemCarveoutMaxShared)) != cudaSuccess) FDAS_CREATE_FAIL(FDAS_ERR_CUDA)
            if ((e = cudaFuncSetAttribute((const void *)p->kernel_thr, cudaFuncAttributePreferredSharedMemoryCarveout,
                                          cudaSharedmemCarveoutMaxShared)) != cudaSuccess) FDAS_CREATE_FAIL(FDAS_ERR_CUDA)
        }
        cudaFuncAttributes fa;
        if ((e = cudaFuncGetAttributes(&fa, (const void *)kern)) != cudaSuccess) FDAS_CREATE_FAIL(FDAS_ERR_CUDA)
        I.regs = fa.numRegs;
        int occ = 0;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)kern, I.threads,
                                                               I.smem_bytes)) != cudaSuccess) FDAS_CREATE_FAIL(FDAS_ERR_CUDA)
        if (occ < 1) { st = FDAS_ERR_UNSUPPORTED; break; }
        // cudaOccupancyMaxActiveBlocksPerMultiprocessor answers 1 for any kernel that uses tensor memory
        // (EIATTR_TCGEN05_1CTA_USED); fdas_kernel3.cuh allocates 128 of the SM's 512 columns per CTA and is
        // built for K3_CTAS_PER_SM_2048 CTAs per SM.  Whether that many really fit is worked out here from the
        // compiled kernels' registers and shared memory and the device's limits, for BOTH kernels that share the
        // grid; if fewer fit (another device, a later edit that costs registers) the persistent grid shrinks with it
        // instead of leaving a third of the CTAs to run as a serial tail, and fdas_info reports the smaller number.
        if (seglen == 2048 && occ < K3_CTAS_PER_SM_2048) {
            cudaFuncAttributes fb;
            if ((e = cudaFuncGetAttributes(&fb, (const void *)p->kernel_thr)) != cudaSuccess) FDAS_CREATE_FAIL(FDAS_ERR_CUDA)
            const int tm = tmem_cols_for(seglen);
            const int fit = std::min(resident_ctas(prop, fa, I.threads, I.smem_bytes, tm),
                                     resident_ctas(prop, fb, I.threads, I.smem_bytes, tm));
            occ = std::max(occ, std::min(fit, K3_CTAS_PER_SM_2048));
        }
        I.ctas_per_sm = occ;
        I.grid = occ * I.sm_count;
        const size_t taps_bytes = (size_t)p->nbanks * K * (2 * m + 1) * sizeof(double2);
        const size_t h_bytes = (size_t)p->nbanks * I.npairs * seglen * sizeof(float2);
        if (cudaMalloc(&p->d_taps, taps_bytes) != cudaSuccess ||
            cudaMalloc(&p->d_hperm, h_bytes) != cudaSuccess ||
            cudaMalloc(&p->d_wtab, (size_t)seglen * sizeof(float2)) != cudaSuccess ||
            (seglen == 8192 && cudaMalloc(&p->d_wtab2, (size_t)seglen * sizeof(float2)) != cudaSuccess)) {
            e = cudaGetLastError();
            FDAS_CREATE_FAIL(FDAS_ERR_NOMEM)
        }
#undef FDAS_CREATE_FAIL
    } while (0);
    if (st != FDAS_OK) {
        fdas_destroy(p);
        return st;
    }
    *out = p;
    return FDAS_OK;
}

fdas_status fdas_make_templates(fdas_plan *p, void *stream)
{
    if (!p || !on_plan_device(p)) return FDAS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const fdas_info &I = p->info;
    const int w = 2 * I.halfwidth + 1;
    {
        const int n = I.ntemplates * w;                      // <= 2e9: checked in fdas_plan_create
        for (int b = 0; b < p->nbanks; ++b)
            make_taps_kernel<<<(n + 127) / 128, 128, 0, st>>>(p->d_taps + (size_t)b * n, I.ntemplates, I.halfwidth,
                                                              I.zmax, I.dz, b);
        g_launches += p->nbanks - 1;
        const int lw = I.seglen == 8192 ? 4096 : I.seglen;   // table of the kernel's passes
        make_wtab_kernel<<<(lw + 127) / 128, 128, 0, st>>>(p->d_wtab, lw);
        if (I.seglen == 8192) {
            make_wtab_kernel<<<(8192 + 127) / 128, 128, 0, st>>>(p->d_wtab2, 8192);
            g_launches += 1;
        }
        const int nh = I.npairs * I.seglen;
        const int gb = (nh + 127) / 128;
        switch (I.seglen) {
        case 1024:
            for (int b = 0; b < p->nbanks; ++b)
                make_spectra_kernel<1024><<<gb, 128, 0, st>>>(p->d_hperm, p->d_taps + (size_t)b * n, I.npairs, I.halfwidth,
                                                            I.zmax, I.dz, I.ntemplates, p->nbanks, b);
            break;
        case 2048:
            for (int b = 0; b < p->nbanks; ++b)
                make_spectra_kernel<2048, 3><<<gb, 128, 0, st>>>(p->d_hperm, p->d_taps + (size_t)b * n, I.npairs, I.halfwidth,
                                                            I.zmax, I.dz, I.ntemplates, p->nbanks, b);
            break;
        case 4096:
            for (int b = 0; b < p->nbanks; ++b)
                make_spectra_kernel<4096><<<gb, 128, 0, st>>>(p->d_hperm, p->d_taps + (size_t)b * n, I.npairs, I.halfwidth,
                                                            I.zmax, I.dz, I.ntemplates, p->nbanks, b);
            break;
        case 8192:
            for (int b = 0; b < p->nbanks; ++b)
                make_spectra_kernel_8k<<<gb, 128, 0, st>>>(p->d_hperm, p->d_taps + (size_t)b * n, I.npairs, I.halfwidth, I.zmax,
                                                           I.dz, I.ntemplates, p->nbanks, b);
            break;
        default: return FDAS_ERR_UNSUPPORTED;
        }
        g_launches += 3;
    }
    FDAS_CUDA(p, cudaGetLastError());
    p->ready = true;
    return FDAS_OK;
}

static fdas_status launch_fused(fdas_plan *p, void *stream, const void *d_spectrum, float *d_plane,
                                float threshold, fdas_candidate *d_cands, int64_t capacity,
                                unsigned long long *d_count)
{
    const fdas_info &I = p->info;
    KernelParams prm;
    prm.spectrum = (const float2 *)d_spectrum;
    prm.plane = d_plane;
    prm.cands = (Candidate *)d_cands;
    prm.count = d_count;
    prm.capacity = capacity;
    prm.threshold = threshold;
    prm.hperm = (const float4 *)p->d_hperm;
    prm.wtab = p->d_wtab;
    prm.wtab2 = p->d_wtab2;
    prm.nbins = I.nbins;
    prm.ncols = I.ncols;
    prm.nseg = I.nseg;
    prm.ntemplates = I.ntemplates;
    prm.npairs = I.npairs * p->nbanks;      // template slots per segment (bank-minor)
    prm.overlap = I.overlap;
    prm.useful = I.useful;
    void *args[] = {&prm};
    const void *kern = d_count ? (const void *)p->kernel_thr : (const void *)p->kernel;
    FDAS_CUDA(p, cudaLaunchKernel(kern, dim3(I.grid), dim3(I.threads), args,
                                  (size_t)I.smem_bytes, (cudaStream_t)stream));
    g_launches += 1;
    return FDAS_OK;
}

fdas_status fdas_execute(fdas_plan *p, void *stream, const void *d_spectrum, float *d_plane)
{
    if (!p || !d_spectrum || !d_plane || !on_plan_device(p)) return FDAS_ERR_INVALID_ARG;
    if (!p->ready) return FDAS_ERR_NOT_READY;
    if (((uintptr_t)d_spectrum & 15) || ((uintptr_t)d_plane & 15)) return FDAS_ERR_ALIGNMENT;
    return launch_fused(p, stream, d_spectrum, d_plane, 0.f, nullptr, 0, nullptr);
}

fdas_status fdas_execute_threshold(fdas_plan *p, void *stream, const void *d_spectrum, float threshold,
                                   fdas_candidate *d_cands, int64_t capacity, uint64_t *d_count)
{
    if (!p || !d_spectrum || !d_count || capacity < 0 || (capacity > 0 && !d_cands) || threshold != threshold ||
        !on_plan_device(p))
        return FDAS_ERR_INVALID_ARG;
    if (!p->ready) return FDAS_ERR_NOT_READY;
    if (((uintptr_t)d_spectrum & 15) || (capacity > 0 && ((uintptr_t)d_cands & 15)) || ((uintptr_t)d_count & 7))
        return FDAS_ERR_ALIGNMENT;   // d_cands is never written when capacity is 0
    FDAS_CUDA(p, cudaMemsetAsync(d_count, 0, sizeof(uint64_t), (cudaStream_t)stream));
    return launch_fused(p, stream, d_spectrum, nullptr, threshold, d_cands, capacity,
                        (unsigned long long *)d_count);
}

fdas_status fdas_execute_host(fdas_plan *p, void *stream, const void *h_spectrum, float *h_plane)
{
    if (!p || !h_spectrum || !h_plane || !on_plan_device(p)) return FDAS_ERR_INVALID_ARG;
    if (!p->ready) return FDAS_ERR_NOT_READY;
    const fdas_info &I = p->info;
    cudaStream_t st = (cudaStream_t)stream;
    // the two staging buffers are allocated independently: fdas_execute_threshold_host shares d_stage_in only
    if (!p->d_stage_in && cudaMalloc(&p->d_stage_in, (size_t)I.nbins * sizeof(float2)) != cudaSuccess) {
        cudaGetLastError();
        p->d_stage_in = nullptr;
        return FDAS_ERR_NOMEM;
    }
    if (!p->d_stage_out && cudaMalloc(&p->d_stage_out, (size_t)I.plane_bytes) != cudaSuccess) {
        cudaGetLastError();
        p->d_stage_out = nullptr;
        return FDAS_ERR_NOMEM;
    }
    FDAS_CUDA(p, cudaMemcpyAsync(p->d_stage_in, h_spectrum, (size_t)I.nbins * sizeof(float2),
                                 cudaMemcpyHostToDevice, st));
    fdas_status s = fdas_execute(p, stream, p->d_stage_in, p->d_stage_out);
    if (s != FDAS_OK) return s;
    FDAS_CUDA(p, cudaMemcpyAsync(h_plane, p->d_stage_out, (size_t)I.plane_bytes, cudaMemcpyDeviceToHost, st));
    FDAS_CUDA(p, cudaStreamSynchronize(st));
    return FDAS_OK;
}

fdas_status fdas_execute_threshold_host(fdas_plan *p, void *stream, const void *h_spectrum, float threshold,
                                        fdas_candidate *h_cands, int64_t capacity, uint64_t *h_count)
{
    if (!p || !h_spectrum || !h_count || capacity < 0 || (capacity > 0 && !h_cands) || !on_plan_device(p))
        return FDAS_ERR_INVALID_ARG;
    if (!p->ready) return FDAS_ERR_NOT_READY;
    const fdas_info &I = p->info;
    cudaStream_t st = (cudaStream_t)stream;
    if (!p->d_stage_in && cudaMalloc(&p->d_stage_in, (size_t)I.nbins * sizeof(float2)) != cudaSuccess) {
        cudaGetLastError();
        return FDAS_ERR_NOMEM;
    }
    if (!p->d_stage_count && cudaMalloc(&p->d_stage_count, sizeof(unsigned long long)) != cudaSuccess) {
        cudaGetLastError();
        return FDAS_ERR_NOMEM;
    }
    if (capacity > p->stage_cands_cap) {
        FDAS_CUDA(p, cudaStreamSynchronize(st));
        cudaFree(p->d_stage_cands);
        p->d_stage_cands = nullptr;
        p->stage_cands_cap = 0;
        if (cudaMalloc(&p->d_stage_cands, (size_t)capacity * sizeof(fdas_candidate)) != cudaSuccess) {
            cudaGetLastError();
            return FDAS_ERR_NOMEM;
        }
        p->stage_cands_cap = capacity;
    }
    FDAS_CUDA(p, cudaMemcpyAsync(p->d_stage_in, h_spectrum, (size_t)I.nbins * sizeof(float2),
                                 cudaMemcpyHostToDevice, st));
    fdas_status s = fdas_execute_threshold(p, stream, p->d_stage_in, threshold, p->d_stage_cands, capacity,
                                           (uint64_t *)p->d_stage_count);
    if (s != FDAS_OK) return s;
    FDAS_CUDA(p, cudaMemcpyAsync(h_count, p->d_stage_count, sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
    FDAS_CUDA(p, cudaStreamSynchronize(st));
    const uint64_t nvalid = *h_count < (uint64_t)capacity ? *h_count : (uint64_t)capacity;
    if (nvalid) {
        FDAS_CUDA(p, cudaMemcpyAsync(h_cands, p->d_stage_cands, (size_t)nvalid * sizeof(fdas_candidate),
                                     cudaMemcpyDeviceToHost, st));
        FDAS_CUDA(p, cudaStreamSynchronize(st));
    }
    return FDAS_OK;
}

fdas_status fdas_harmonic_sum_threshold(fdas_plan *p, void *stream, const float *d_plane, int32_t nharm,
                                        float threshold, fdas_candidate *d_cands, int64_t capacity, uint64_t *d_count)
{
    if (!p || !d_plane || !d_count || nharm < 1 || capacity < 0 || (capacity > 0 && !d_cands) ||
        threshold != threshold || !on_plan_device(p))
        return FDAS_ERR_INVALID_ARG;
    if (((uintptr_t)d_plane & 15) || (capacity > 0 && ((uintptr_t)d_cands & 15)) || ((uintptr_t)d_count & 7))
        return FDAS_ERR_ALIGNMENT;
    const fdas_info &I = p->info;
    cudaStream_t st = (cudaStream_t)stream;
    FDAS_CUDA(p, cudaMemsetAsync(d_count, 0, sizeof(uint64_t), st));
    const int nhalf = (I.ntemplates - 1) / 2, lim = nhalf / nharm;      // rows |z_k| <= zmax / H
    const long long nc = (I.ncols - 1) / nharm + 1;
    // one CTA per (row, block of 1024 columns), rows folded into blockIdx.x: grid.y would cap the bank at 65 535 rows
    const long long nbx = (nc + 1023) / 1024, nblocks = nbx * (2 * lim + 1);    // 4 columns per thread
    if (nblocks > 0x7fffffffll) {
        snprintf(p->err, sizeof(p->err), "fdas_harmonic_sum_threshold: %lld CTAs exceed the grid limit", nblocks);
        return FDAS_ERR_UNSUPPORTED;
    }
    harmonic_sum_kernel<<<(unsigned)nblocks, 256, 0, st>>>(d_plane, I.ncols, I.ntemplates, nharm, nhalf - lim,
                                                           (unsigned)nbx, threshold, (Candidate *)d_cands, capacity,
                                                           (unsigned long long *)d_count);
    g_launches += 1;
    FDAS_CUDA(p, cudaGetLastError());
    return FDAS_OK;
}

fdas_status fdas_harmonic_sums_threshold(fdas_plan *p, void *stream, const float *d_plane, int32_t nlevels,
                                         const int32_t *nharm, const float *thresholds, fdas_candidate *d_cands,
                                         int64_t capacity, uint64_t *d_counts)
{
    if (!p || !d_plane || !d_counts || !nharm || !thresholds || nlevels < 1 || nlevels > 4 || capacity < 0 ||
        (capacity > 0 && !d_cands) || !on_plan_device(p))
        return FDAS_ERR_INVALID_ARG;
    HarmonicLevels lv;
    std::memset(&lv, 0, sizeof(lv));
    for (int l = 0; l < nlevels; ++l) {
        if (nharm[l] < 1 || (l > 0 && nharm[l] <= nharm[l - 1]) || thresholds[l] != thresholds[l])
            return FDAS_ERR_INVALID_ARG;
        lv.nharm[l] = nharm[l];
        lv.threshold[l] = thresholds[l];
    }
    if (((uintptr_t)d_plane & 15) || (capacity > 0 && ((uintptr_t)d_cands & 15)) || ((uintptr_t)d_counts & 7))
        return FDAS_ERR_ALIGNMENT;
    const fdas_info &I = p->info;
    cudaStream_t st = (cudaStream_t)stream;
    FDAS_CUDA(p, cudaMemsetAsync(d_counts, 0, sizeof(uint64_t) * nlevels, st));
    lv.nlevels = nlevels;
    lv.capacity = capacity;
    lv.cands = (Candidate *)d_cands;
    lv.counts = (unsigned long long *)d_counts;
    const int nhalf = (I.ntemplates - 1) / 2, lim = nhalf / nharm[0];       // the first level has the widest domain
    const long long nc = (I.ncols - 1) / nharm[0] + 1;
    const long long nbx = (nc + 1023) / 1024, nblocks = nbx * (2 * lim + 1);
    if (nblocks > 0x7fffffffll) {
        snprintf(p->err, sizeof(p->err), "fdas_harmonic_sums_threshold: %lld CTAs exceed the grid limit", nblocks);
        return FDAS_ERR_UNSUPPORTED;
    }
    harmonic_sums_kernel<<<(unsigned)nblocks, 256, 0, st>>>(d_plane, I.ncols, I.ntemplates, (unsigned)nbx, lv);
    g_launches += 1;
    FDAS_CUDA(p, cudaGetLastError());
    return FDAS_OK;
}

fdas_status fdas_destroy(fdas_plan *p)
{
    if (!p) return FDAS_OK;
    cudaFree(p->d_stage_cands);
    cudaFree(p->d_stage_count);
    cudaFree(p->d_taps);
    cudaFree(p->d_hperm);
    cudaFree(p->d_wtab);
    cudaFree(p->d_wtab2);
    cudaFree(p->d_stage_in);
    cudaFree(p->d_stage_out);
    cudaGetLastError();
    delete p;
    return FDAS_OK;
}

fdas_status fdas_plan_info(const fdas_plan *p, fdas_info *out)
{
    if (!p || !out) return FDAS_ERR_INVALID_ARG;
    *out = p->info;
    return FDAS_OK;
}

fdas_status fdas_get_taps(fdas_plan *p, int32_t k, double *host_re_im, int32_t *halfwidth_k)
{
    if (!p || !host_re_im || !halfwidth_k || k < 0 || k >= p->info.ntemplates * p->nbanks || !on_plan_device(p))
        return FDAS_ERR_INVALID_ARG;
    if (!p->ready) return FDAS_ERR_NOT_READY;
    const fdas_info &I = p->info;
    const int m = I.halfwidth, w = 2 * m + 1;
    const int kk = k % I.ntemplates;            // k >= ntemplates: bank 1 (interbin = 2), taps h_z(d - 1/2)
    const int center = (I.ntemplates - 1) / 2;
    const double z = (kk == center) ? 0.0 : -I.zmax + kk * I.dz;
    const int mz = (int)std::ceil(std::fabs(z) * 0.5 - 1e-12) + 16;
    FDAS_CUDA(p, cudaDeviceSynchronize());
    FDAS_CUDA(p, cudaMemcpy(host_re_im, p->d_taps + (size_t)k * w + (m - mz),
                            (size_t)(2 * mz + 1) * sizeof(double2), cudaMemcpyDeviceToHost));
    *halfwidth_k = mz;
    return FDAS_OK;
}

fdas_status fdas_get_template_spectrum(fdas_plan *p, int32_t k, float *host_re_im)
{
    if (!p || !host_re_im || k < 0 || k >= p->info.ntemplates || !on_plan_device(p)) return FDAS_ERR_INVALID_ARG;
    if (!p->ready) return FDAS_ERR_NOT_READY;
    const fdas_info &I = p->info;
    const int L = I.seglen, T = I.threads;
    const int pair = k < I.ntemplates - 1 - k ? k : I.ntemplates - 1 - k;
    const bool conj = k != pair;
    std::vector<float2> buf(L);
    FDAS_CUDA(p, cudaDeviceSynchronize());
    FDAS_CUDA(p, cudaMemcpy(buf.data(), p->d_hperm + (size_t)pair * p->nbanks * L, (size_t)L * sizeof(float2),
                            cudaMemcpyDeviceToHost));
    for (int f = 0; f < L; ++f) {
        int tid, i;
        freq_to_reg_any(L, f, tid, i);
        const size_t half = (L == 8192) ? (size_t)(f >> 12) * 4096 : 0;   // [half][i/2][tid]
        const float2 v = buf[half + ((size_t)(i >> 1) * T + tid) * 2 + (i & 1)];
        host_re_im[2 * f] = v.x;
        host_re_im[2 * f + 1] = conj ? -v.y : v.y; // H_{+z} = conj(H_{-z})
    }
    return FDAS_OK;
}

// ---------------------------------------------------------------- real-to-complex transform (fdas_r2c.cuh)
} // extern "C"

constexpr int R2C_THREADS = 512;

struct fdas_r2c_plan {
    int64_t n, M;
    int device;
    int lg[3];           // log2 of N1, N2, N3
    int lt[3];           // log2 of the transforms per CTA in passes A, B, C
    float2 *d_work[2], *d_w[3], *d_tlo, *d_thi;
};

extern "C" {

fdas_status fdas_r2c_plan_create(fdas_r2c_plan **out, int64_t nsamples)
{
    if (!out) return FDAS_ERR_INVALID_ARG;
    *out = nullptr;
    if (nsamples <= 0) return FDAS_ERR_INVALID_ARG;
    int p2 = 0;
    while ((1ll << p2) < nsamples) ++p2;
    if ((1ll << p2) != nsamples || p2 < 10 || p2 > 25) return FDAS_ERR_UNSUPPORTED;
    fdas_r2c_plan *p = new (std::nothrow) fdas_r2c_plan();
    if (!p) return FDAS_ERR_NOMEM;
    std::memset(p, 0, sizeof(*p));
    p->n = nsamples;
    p->M = nsamples / 2;
    const int lm = p2 - 1;                               // M = N1 N2 N3, factors as equal as possible (<= 2^8)
    p->lg[0] = lm / 3;
    p->lg[1] = (lm - p->lg[0]) / 2;
    p->lg[2] = lm - p->lg[0] - p->lg[1];
    // transforms per CTA: 32 (one warp of columns), fewer where a dimension is shorter; <= 8192 points per CTA
    auto ltile_for = [](int log2R, int log2avail) {
        int t = 5;
        if (t > log2avail) t = log2avail;
        if (t > 13 - log2R) t = 13 - log2R;
        return t;
    };
    p->lt[0] = ltile_for(p->lg[0], p->lg[1] + p->lg[2]);
    p->lt[1] = ltile_for(p->lg[1], p->lg[2]);
    p->lt[2] = ltile_for(p->lg[2], p->lg[0]);
    g_create_err[0] = 0;
    const int64_t nhi = (nsamples + 4095) / 4096;
    cudaError_t e = cudaGetDevice(&p->device);
    for (int i = 0; i < 2; ++i)
        if (e == cudaSuccess) e = cudaMalloc(&p->d_work[i], (size_t)p->M * sizeof(float2));
    for (int i = 0; i < 3; ++i)
        if (e == cudaSuccess) e = cudaMalloc(&p->d_w[i], (sizeof(float2)) << p->lg[i]);
    if (e == cudaSuccess) e = cudaMalloc(&p->d_tlo, 4096 * sizeof(float2));
    if (e == cudaSuccess) e = cudaMalloc(&p->d_thi, (size_t)nhi * sizeof(float2));
    if (e == cudaSuccess) {
        for (int i = 0; i < 3; ++i) {
            const long long R = 1ll << p->lg[i];
            r2c_table_kernel<<<(unsigned)((R + 127) / 128), 128>>>(p->d_w[i], R, 1, R);
        }
        r2c_table_kernel<<<32, 128>>>(p->d_tlo, 4096, 1, nsamples);
        r2c_table_kernel<<<(unsigned)((nhi + 127) / 128), 128>>>(p->d_thi, nhi, 4096, nsamples);
        g_launches += 5;
        e = cudaDeviceSynchronize();
    }
    for (const void *k : {(const void *)r2c_cols_kernel, (const void *)r2c_rows_kernel})
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (8192 + 32 + 256) * 8);
    if (e != cudaSuccess) {
        snprintf(g_create_err, sizeof(g_create_err), "fdas_r2c_plan_create: %s", cudaGetErrorString(e));
        const bool nomem = e == cudaErrorMemoryAllocation;
        cudaGetLastError();
        fdas_r2c_destroy(p);
        return nomem ? FDAS_ERR_NOMEM : FDAS_ERR_CUDA;
    }
    *out = p;
    return FDAS_OK;
}

fdas_status fdas_r2c_execute(fdas_r2c_plan *p, void *stream, const float *d_timeseries, void *d_spectrum, float scale)
{
    if (!p || !d_timeseries || !d_spectrum) return FDAS_ERR_INVALID_ARG;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device) return FDAS_ERR_INVALID_ARG;
    if (((uintptr_t)d_timeseries & 7) || ((uintptr_t)d_spectrum & 15)) return FDAS_ERR_ALIGNMENT;
    cudaStream_t st = (cudaStream_t)stream;
    const long long N1 = 1ll << p->lg[0], N2 = 1ll << p->lg[1], N3 = 1ll << p->lg[2];
    auto smem = [](int lg, int lt) { return ((((size_t)1 << lg) + 1) << lt) * sizeof(float2) + (sizeof(float2) << lg); };
    R2CParams q;
    q.tlo = p->d_tlo;
    q.thi = p->d_thi;
    q.M = p->M;
    q.N1 = (int)N1;
    q.N2 = (int)N2;
    q.scale = scale;
    // pass A: length N1 over j1, columns j' = j2 N3 + j3
    q.in = (const float2 *)d_timeseries;
    q.out = p->d_work[0];
    q.wR = p->d_w[0];
    q.log2R = p->lg[0];
    q.ltile = p->lt[0];
    q.inner = N2 * N3;
    q.slab = p->M;
    q.tmul = 2;
    r2c_cols_kernel<<<dim3((unsigned)((N2 * N3) >> p->lt[0]), 1), R2C_THREADS, smem(p->lg[0], p->lt[0]), st>>>(q);
    // pass B: per k1, length N2 over j2, columns j3
    q.in = p->d_work[0];
    q.out = p->d_work[1];
    q.wR = p->d_w[1];
    q.log2R = p->lg[1];
    q.ltile = p->lt[1];
    q.inner = N3;
    q.slab = N2 * N3;
    q.tmul = 2 * N1;
    r2c_cols_kernel<<<dim3((unsigned)(N3 >> p->lt[1]), (unsigned)N1), R2C_THREADS, smem(p->lg[1], p->lt[1]), st>>>(q);
    // pass C: length N3 over j3, transposed store
    q.in = p->d_work[1];
    q.out = (float2 *)d_spectrum;
    q.wR = p->d_w[2];
    q.log2R = p->lg[2];
    q.ltile = p->lt[2];
    q.inner = N3;
    r2c_rows_kernel<<<dim3((unsigned)(N1 >> p->lt[2]), (unsigned)N2), R2C_THREADS, smem(p->lg[2], p->lt[2]), st>>>(q);
    r2c_untangle_kernel<<<(unsigned)((p->M / 2 + 1 + 255) / 256), 256, 0, st>>>(q);
    g_launches += 4;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {                                   // the r2c plan has no text buffer: fdas_last_error(NULL)
        snprintf(g_create_err, sizeof(g_create_err), "fdas_r2c_execute: %s", cudaGetErrorString(e));
        return FDAS_ERR_CUDA;
    }
    return FDAS_OK;
}

fdas_status fdas_r2c_destroy(fdas_r2c_plan *p)
{
    if (!p) return FDAS_OK;
    for (int i = 0; i < 2; ++i) cudaFree(p->d_work[i]);
    for (int i = 0; i < 3; ++i) cudaFree(p->d_w[i]);
    cudaFree(p->d_tlo);
    cudaFree(p->d_thi);
    cudaGetLastError();
    delete p;
    return FDAS_OK;
}

// ---------------------------------------------------------------- red-noise removal / block normalisation (fdas_whiten.cuh)
fdas_status fdas_whiten(void *stream, const void *d_spectrum, void *d_out, int64_t nbins, int32_t block,
                        int32_t statistic)
{
    if (!d_spectrum || !d_out || nbins <= 0 || (statistic != FDAS_WHITEN_MEDIAN && statistic != FDAS_WHITEN_MEAN))
        return FDAS_ERR_INVALID_ARG;
    const long long nblocks = block > 0 ? (nbins + block - 1) / block : 0;
    if (block < WHITEN_MIN_BLOCK || block > WHITEN_MAX_BLOCK || nblocks > 0x7fffffffll) {
        snprintf(g_create_err, sizeof(g_create_err), "fdas_whiten: block = %d, nbins = %lld; needs %d <= block <= %d and at "
                 "most 2^31 - 1 blocks", (int)block, (long long)nbins, WHITEN_MIN_BLOCK, WHITEN_MAX_BLOCK);
        return FDAS_ERR_UNSUPPORTED;
    }
    if (((uintptr_t)d_spectrum & 7) || ((uintptr_t)d_out & 7)) return FDAS_ERR_ALIGNMENT;
    whiten_kernel<<<(unsigned)nblocks, WHITEN_THREADS, whiten_smem_bytes(block), (cudaStream_t)stream>>>(
        (const float2 *)d_spectrum, (float2 *)d_out, nbins, block, statistic);
    g_launches += 1;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(g_create_err, sizeof(g_create_err), "fdas_whiten: %s", cudaGetErrorString(e));
        return FDAS_ERR_CUDA;
    }
    return FDAS_OK;
}

// ---------------------------------------------------------------- the transform for callers that may not allocate
} // extern "C"

// fdas_r2c_execute_static (include/fdas.h) is for hosts that cannot call cudaMalloc while they run: an acquisition
// back-end that divided the card's memory once at start-up and must not take the allocator's device-wide lock (or
// its failure when a neighbour has filled the card) inside its real-time loop, or a plug-in living inside a
// framework whose own pool already holds nearly all of HBM.  For them everything the transform needs beyond its
// input and output -- the two work arrays between the passes and the five twiddle tables -- lives in ONE
// file-scope device array, which every GPU that loads libfdas.so holds from module load until the process exits
// (8.04 MiB; nothing is ever freed).  Layout in float2 elements:
//     [0, MAXM) work 0 | [MAXM, 2 MAXM) work 1 | 3 x 256 exp(-2 pi i j / N_i) | 4096 t_lo | 256 t_hi
// Every sub-array starts on a 256-byte boundary.  Host code may not hand `g_r2c_static_scratch` itself to a
// kernel: on the host that name is only a handle for the symbol; its device address comes from
// cudaGetSymbolAddress, taken once per device (below) with that device current.
constexpr long long R2C_STATIC_MAXM = FDAS_R2C_STATIC_MAX_SAMPLES / 2;
constexpr long long R2C_STATIC_ELEMS = 2 * R2C_STATIC_MAXM + 3 * 256 + 4096 + FDAS_R2C_STATIC_MAX_SAMPLES / 4096;
static __device__ __align__(256) float2 g_r2c_static_scratch[R2C_STATIC_ELEMS];
static_assert(sizeof(float2) * R2C_STATIC_ELEMS == FDAS_R2C_STATIC_BYTES, "fdas.h states the size of the static scratch array");

namespace {

constexpr int R2C_STATIC_MAX_DEVICES = 64;

struct R2CStaticDevice {
    bool ready;            // address taken and kernel attributes set on this device
    fdas_r2c_plan plan;    // a plan whose pointers all lie inside g_r2c_static_scratch; plan.n = size of the tables
};
R2CStaticDevice g_r2c_static_dev[R2C_STATIC_MAX_DEVICES];   // zero-initialised
std::mutex g_r2c_static_mutex;

} // namespace

extern "C" {

fdas_status fdas_r2c_execute_static(void *stream, const float *d_timeseries, int64_t nsamples, void *d_spectrum,
                                    float scale)
{
    if (!d_timeseries || !d_spectrum || nsamples <= 0) return FDAS_ERR_INVALID_ARG;
    int p2 = 0;
    while (p2 < 62 && (1ll << p2) < nsamples) ++p2;
    if ((1ll << p2) != nsamples || p2 < 10 || nsamples > FDAS_R2C_STATIC_MAX_SAMPLES) {
        snprintf(g_create_err, sizeof(g_create_err),
                 "fdas_r2c_execute_static: nsamples = %lld; needs a power of two in [1024, %lld] (the static scratch "
                 "array holds no more; longer series need fdas_r2c_plan_create)",
                 (long long)nsamples, (long long)FDAS_R2C_STATIC_MAX_SAMPLES);
        return FDAS_ERR_UNSUPPORTED;
    }
    if (((uintptr_t)d_timeseries & 7) || ((uintptr_t)d_spectrum & 15)) return FDAS_ERR_ALIGNMENT;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess && (dev < 0 || dev >= R2C_STATIC_MAX_DEVICES)) {
        snprintf(g_create_err, sizeof(g_create_err), "fdas_r2c_execute_static: device ordinal %d not supported", dev);
        return FDAS_ERR_UNSUPPORTED;
    }
    if (e != cudaSuccess) {
        snprintf(g_create_err, sizeof(g_create_err), "fdas_r2c_execute_static: %s", cudaGetErrorString(e));
        cudaGetLastError();
        return FDAS_ERR_CUDA;
    }
    cudaStream_t st = (cudaStream_t)stream;
    std::lock_guard<std::mutex> lock(g_r2c_static_mutex);
    R2CStaticDevice &D = g_r2c_static_dev[dev];
    fdas_r2c_plan &P = D.plan;
    if (!D.ready) {
        // Once per device, with that device current: the array's address ON THIS DEVICE, and the shared-memory
        // limit of the two transform kernels (a per-device function attribute).  Neither allocates.
        float2 *base = nullptr;
        e = cudaGetSymbolAddress((void **)&base, g_r2c_static_scratch);
        for (const void *k : {(const void *)r2c_cols_kernel, (const void *)r2c_rows_kernel})
            if (e == cudaSuccess)
                e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (8192 + 32 + 256) * 8);
        if (e != cudaSuccess || !base) {
            snprintf(g_create_err, sizeof(g_create_err), "fdas_r2c_execute_static: set-up on device %d: %s", dev,
                     e != cudaSuccess ? cudaGetErrorString(e) : "null symbol address");
            cudaGetLastError();
            return FDAS_ERR_CUDA;
        }
        std::memset(&P, 0, sizeof(P));
        P.device = dev;
        P.d_work[0] = base;
        P.d_work[1] = base + R2C_STATIC_MAXM;
        for (int i = 0; i < 3; ++i) P.d_w[i] = base + 2 * R2C_STATIC_MAXM + 256 * i;
        P.d_tlo = P.d_w[2] + 256;
        P.d_thi = P.d_tlo + 4096;
        D.ready = true;
    }
    if (P.n != nsamples) {
        // Another length than the last call on this device: same factorisation rule as fdas_r2c_plan_create, and
        // the tables are refilled ON THE CALLER'S STREAM, behind whatever that stream still has to do with the old
        // ones.  (The work arrays need no clearing: every pass writes all M elements before the next reads them.)
        const int lm = p2 - 1;
        P.lg[0] = lm / 3;
        P.lg[1] = (lm - P.lg[0]) / 2;
        P.lg[2] = lm - P.lg[0] - P.lg[1];
        auto ltile_for = [](int log2R, int log2avail) {
            int t = 5;
            if (t > log2avail) t = log2avail;
            if (t > 13 - log2R) t = 13 - log2R;
            return t;
        };
        P.lt[0] = ltile_for(P.lg[0], P.lg[1] + P.lg[2]);
        P.lt[1] = ltile_for(P.lg[1], P.lg[2]);
        P.lt[2] = ltile_for(P.lg[2], P.lg[0]);
        P.n = 0;                                              // tables invalid until all five launches are queued
        P.M = nsamples / 2;
        const long long nhi = (nsamples + 4095) / 4096;
        for (int i = 0; i < 3; ++i) {
            const long long R = 1ll << P.lg[i];
            r2c_table_kernel<<<(unsigned)((R + 127) / 128), 128, 0, st>>>(P.d_w[i], R, 1, R);
        }
        r2c_table_kernel<<<32, 128, 0, st>>>(P.d_tlo, 4096, 1, nsamples);
        r2c_table_kernel<<<(unsigned)((nhi + 127) / 128), 128, 0, st>>>(P.d_thi, nhi, 4096, nsamples);
        g_launches += 5;
        e = cudaGetLastError();
        if (e != cudaSuccess) {
            snprintf(g_create_err, sizeof(g_create_err), "fdas_r2c_execute_static: twiddle tables: %s",
                     cudaGetErrorString(e));
            return FDAS_ERR_CUDA;
        }
        P.n = nsamples;
    }
    return fdas_r2c_execute(&P, stream, d_timeseries, d_spectrum, scale);   // the four passes, unchanged
}

fdas_status fdas_measure_fp32_peak(void *stream, int32_t iters, double *tflops)
{
    if (!tflops || iters <= 0) return FDAS_ERR_INVALID_ARG;
    *tflops = 0.0;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    float *d_out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    fdas_status rc = FDAS_ERR_CUDA;
    do {
        if (cudaGetDevice(&dev) != cudaSuccess) break;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) break;
        if (cudaMalloc(&d_out, 4) != cudaSuccess) break;
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) break;
        const int grid = sms * 8, block = 256;
        fp32_peak_kernel<<<grid, block, 0, st>>>(d_out, 16, 1.0001f, 0.5f); // warm-up
        cudaEventRecord(e0, st);
        fp32_peak_kernel<<<grid, block, 0, st>>>(d_out, iters, 1.0001f, 0.5f);
        cudaEventRecord(e1, st);
        g_launches += 2;
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) break;
        const double flops = 2.0 * 8.0 * 16.0 * (double)iters * (double)grid * block;
        *tflops = flops / (ms * 1e-3) / 1e12;
        rc = FDAS_OK;
    } while (0);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(d_out);
    return rc;
}

} // extern "C"
