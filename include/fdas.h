/*
 * fdas.h -- C ABI of the B200-native FDAS correlation hot path (arXiv:1804.05335).
 *
 * The library computes the f-fdot power plane of the paper's "correlation technique":
 * the overlap-save convolution of a complex Fourier spectrum with a bank of
 * per-trial-z Fourier-domain FIR templates, followed by |.|^2 (optionally interbinned).
 * Citations are to /root/reference/PAPER.md (line numbers) and to DESIGN.md readings (Rn).
 *
 *   result (eq. 3):
 *       y_z[r] = sum_{d=-m_z}^{+m_z} A[r+d] * conj(h_z[d]),  A[j] := 0 outside [0, nbins)
 *       P[z][r] = |y_z[r]|^2
 *   method (PAPER.md:75-77, :87 Fig. 1, :105, :129-131): per overlapping segment of
 *       `seglen` bins: forward FFT, pointwise multiply by each template's precomputed
 *       FFT, inverse FFT, discard the contaminated edges, power, contiguous store.
 *   interbinning (PAPER.md:81-83 eq. 4, :89, :95), applied to the correlated amplitudes:
 *       P[z][2r] = |y_z[r]|^2,  P[z][2r+1] = |(pi/4)(y_z[r] - y_z[r+1])|^2
 *   two-bin Fourier interpolation ("doubling the template and signal resolution using
 *   interleaving zeros prior to the correlations"; reading R16), the accurate alternative:
 *       P[z][2r] = |y_z[r]|^2,  P[z][2r+1] = |sum_{d=-m_z+1}^{m_z} A[r+d] * conj(h_z(d - 1/2))|^2
 *
 * All entry points are plain C, take plain pointers and sizes, return a status code and
 * never throw or abort.  "device" pointers are CUDA device pointers on the device that
 * was current when the plan was created; every call that takes a plan returns
 * FDAS_ERR_INVALID_ARG when another device is current.  "host" pointers are ordinary host memory.
 * `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 * There is no CPU fallback anywhere in this library.
 */
#ifndef FDAS_H_
#define FDAS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fdas_plan fdas_plan; /* opaque; created/destroyed by the library */

typedef enum fdas_status {
    FDAS_OK = 0,
    FDAS_ERR_INVALID_ARG = 1, /* null pointer, nbins <= 0, zmax < 0, dz <= 0, zmax/dz not an integer      */
    FDAS_ERR_UNSUPPORTED = 2, /* seglen not in {1024, 2048, 4096, 8192}, or too short for the bank's overlap,
                                 or a bank beyond 2e9 taps / spectrum slots                                   */
    FDAS_ERR_NOT_READY = 3,   /* fdas_execute before fdas_make_templates                                    */
    FDAS_ERR_ALIGNMENT = 4,   /* device pointer not 16-byte aligned                                         */
    FDAS_ERR_CUDA = 5,        /* a CUDA runtime call failed; see fdas_last_error()                          */
    FDAS_ERR_NOMEM = 6        /* host or device allocation failed                                           */
} fdas_status;

/* Geometry of a plan (filled by fdas_plan_info). */
typedef struct fdas_info {
    int64_t nbins;        /* N: complex bins in the spectrum                                         */
    int64_t ncols;        /* plane columns: N, or 2N when interbinned                                */
    int64_t row_stride;   /* floats between consecutive rows of the plane (= ncols)                  */
    int64_t nseg;         /* overlap-save segments: ceil(N / useful)                                 */
    int64_t plane_bytes;  /* ntemplates * ncols * 4                                                  */
    double zmax, dz;      /* bank: z_k = -zmax + k*dz, k = 0..ntemplates-1 (ascending, R9)           */
    int32_t ntemplates;   /* K = 2*zmax/dz + 1                                                       */
    int32_t seglen;       /* L: segment FFT length                                                   */
    int32_t halfwidth;    /* m = ceil(zmax/2) + 16: half-width of the widest template (R4)           */
    int32_t overlap;      /* bins discarded at each end of a segment (>= m, +1 with interbinning;
                             rounded up to a multiple of 32 so segment loads/stores stay 128B-aligned) */
    int32_t useful;       /* B = L - 2*overlap useful output bins per segment                        */
    int32_t interbin;     /* 0 none, 1 interbinning (eq. 4), 2 two-bin Fourier interpolation         */
    int32_t npairs;       /* (K+1)/2 template slots processed by the kernel (+-z share one slot)      */
    int32_t threads;      /* threads per CTA of the fused kernel                                     */
    int32_t grid;         /* CTAs launched by fdas_execute (persistent; multiple of the SM count)    */
    int32_t ctas_per_sm;  /* resident CTAs per SM the grid was sized for: the occupancy API's answer, or, for
                             the tensor-memory kernel of seglen 2048 (where that API answers 1), the number
                             worked out from the compiled kernels' registers and shared memory and the
                             device's limits (3 on a B200; smaller if fewer fit, never assumed)          */
    int32_t smem_bytes;   /* dynamic shared memory per CTA                                           */
    int32_t regs;         /* registers per thread of the fused kernel                                */
    int32_t sm_count;     /* SMs on the device                                                       */
    int32_t reserved;
} fdas_info;

/*
 * Create a plan for spectra of `nbins` complex64 bins and the template bank
 * z = -zmax .. +zmax step dz ("K acceleration templates"; BASELINE.json),
 * each template of half-width ceil(|z|/2)+16 bins (R4), segment FFT length `seglen`
 * ("blocks of length L"); `interbin` = 0: N columns; 1: 2N columns, half-bin cells
 * by interbinning (eq. 4), any seglen; 2: 2N columns, half-bin cells by two-bin
 * Fourier interpolation (a second template bank, twice the transforms), any seglen.
 * Allocates the plan-owned device memory (taps, template spectra, twiddle table).
 * *out is set to NULL on failure.
 * Debug aid: with the environment variable FDAS_DEBUG_E1_SYNC=1 at the time of this call, a seglen-8192 plan's
 * fdas_execute runs a build of its kernel with a CTA barrier in front of every store into the shared exchange
 * buffer (the hand-shake the shipped kernel replaces by an ordering argument).  Same bits, a few per cent slower;
 * a difference between the two planes points at a race in the shipped kernel.
 */
fdas_status fdas_plan_create(fdas_plan **out, int64_t nbins, double zmax, double dz,
                             int32_t seglen, int32_t interbin);

/*
 * Generate the template bank on the device, enqueued on `stream` (no host sync):
 *  a0  taps h_z[d], |d| <= m_z: the "predicted normalised Fourier response",
 *      Fresnel-integral closed form of  int_0^1 exp(2 pi i[-d u + z(u^2-u)/2]) du  (R1), fp64;
 *  a1  template spectra H_z = (1/L) DFT_L(g_z), g_z[j mod L] = conj(h_z[-j]) -- the filter
 *      "centered at bin zero", halves at both ends of an L-array, zeros between
 *      (PAPER.md:77, :87), evaluated in fp64, stored as complex64 in the fused kernel's
 *      un-permuted FFT order; only z <= 0 is stored, +z is applied as
 *      the complex conjugate.  1/L of eq. 6 is folded in (R6).
 */
fdas_status fdas_make_templates(fdas_plan *plan, void *stream);

/*
 * Compute the f-fdot plane of one spectrum: one fused kernel launch on `stream`.
 *   d_spectrum : device, nbins x {float re, float im} (complex64), 16-byte aligned; read only.
 *   d_plane    : device, ntemplates x ncols float32, row-major, 16-byte aligned; every
 *                element is written.  Row k <-> z_k ascending; column r <-> bin r
 *                (interbinned: column 2r <-> bin r, 2r+1 <-> bin r + 1/2).
 * Allocates nothing, never synchronises the host, may be called repeatedly (e.g. once per
 * spectrum of a batch on one stream).  Caller owns both buffers.
 */
fdas_status fdas_execute(fdas_plan *plan, void *stream, const void *d_spectrum, float *d_plane);

/*
 * End-to-end convenience for HOST buffers: copies `h_spectrum` (nbins complex64) to a
 * plan-owned device buffer, runs fdas_execute, copies the plane back to `h_plane`
 * (ntemplates x ncols float32) and synchronises `stream`.  Device staging buffers are
 * allocated on first use and freed by fdas_destroy.  Pinned host memory is recommended.
 */
fdas_status fdas_execute_host(fdas_plan *plan, void *stream, const void *h_spectrum, float *h_plane);

/*
 * One cell of the plane above the threshold (16 bytes).
 */
typedef struct fdas_candidate {
    int64_t col;    /* plane column (0..ncols-1; interbinned: 2r <-> bin r, 2r+1 <-> bin r + 1/2) */
    int32_t row;    /* template row k <-> z_k = -zmax + k*dz                                       */
    float power;    /* P[row][col], the value fdas_execute would have stored                       */
} fdas_candidate;

/*
 * Threshold search fused behind the power step ("calculating the power spectrum,
 * and comparing the resulting Fourier power to a pre-calculated threshold"; PAPER.md:331 names
 * search / candidate selection on on-chip data as the step to fuse next; reading R15).
 * Runs the same fused kernel as fdas_execute (steps a2-a7) but the plane is never written:
 * every cell with P > threshold (strict; NaN never passes) is appended to `d_cands`.
 *   d_spectrum : as for fdas_execute.
 *   d_cands    : device, `capacity` entries, 16-byte aligned (may be NULL when capacity = 0).
 *   d_count    : device, one uint64, 8-byte aligned; zeroed on `stream` by this call, then
 *                incremented once per cell found.  *d_count may exceed `capacity`: only the
 *                first min(*d_count, capacity) entries of d_cands are valid, in no defined
 *                order (sort on (row, col) to compare), and WHICH cells were dropped when it
 *                overflows is unspecified.
 * Allocates nothing, never synchronises the host.  Errors as fdas_execute, plus
 * FDAS_ERR_INVALID_ARG for a NaN threshold, capacity < 0 or a NULL d_count.
 */
fdas_status fdas_execute_threshold(fdas_plan *plan, void *stream, const void *d_spectrum, float threshold,
                                   fdas_candidate *d_cands, int64_t capacity, uint64_t *d_count);

/*
 * End-to-end threshold search for HOST buffers: copies `h_spectrum` to a plan-owned device buffer,
 * runs fdas_execute_threshold, copies the count to *h_count, then the first min(*h_count, capacity)
 * candidates to `h_cands`, and synchronises `stream`.  Staging buffers are allocated on first use
 * (the candidate buffer grows when `capacity` does) and freed by fdas_destroy.
 */
fdas_status fdas_execute_threshold_host(fdas_plan *plan, void *stream, const void *h_spectrum, float threshold,
                                        fdas_candidate *h_cands, int64_t capacity, uint64_t *h_count);

/*
 * Harmonic summing of a stored plane with a threshold search on the sums ("harmonic summing",
 * :79 Fig. 2, :331; reading R18).  A signal whose fundamental sits at plane column c with drift z_k has
 * its h-th harmonic at column h*c with drift h*z_k, so
 *     S_H[k][c] = sum_{h=1}^{H} P[row(h z_k)][h c]
 * is formed for the rows with |z_k| <= zmax / H (all H harmonics inside the bank) and the columns with
 * H*c <= ncols - 1, and every cell with S_H > threshold (strict) is appended to `d_cands` as
 * {col = c, row = k (bank row of the fundamental), power = S_H}.  nharm = 1 is the plain threshold search of a
 * stored plane.  One launch on `stream`; allocates nothing, never synchronises the host.
 *   d_plane : device, the ntemplates x ncols float32 plane fdas_execute wrote (read only), 16-byte aligned.
 *   nharm   : H >= 1 (searches usually sum 2, 4, 8, 16 harmonics in turn; call once per H).
 *   d_cands / capacity / d_count : as for fdas_execute_threshold (d_count is zeroed on `stream` first).
 * Errors: FDAS_ERR_INVALID_ARG (null pointers, nharm < 1, NaN threshold, capacity < 0), FDAS_ERR_ALIGNMENT (d_cands
 * is checked only when capacity > 0: it is never written otherwise), FDAS_ERR_UNSUPPORTED (rows x ceil(columns /
 * 1024) beyond 2^31 - 1 CTAs; any bank size is fine otherwise), FDAS_ERR_CUDA.  Needs no templates (works on any
 * plane of the plan's shape).
 */
fdas_status fdas_harmonic_sum_threshold(fdas_plan *plan, void *stream, const float *d_plane, int32_t nharm,
                                        float threshold, fdas_candidate *d_cands, int64_t capacity,
                                        uint64_t *d_count);

/*
 * The harmonic search for several H in one pass ("adding the power that is distributed in the harmonics to
 * that of the fundamental", :331; reading R18): for the increasing list nharm[0..nlevels) (usually 2, 4, 8, 16) the sums
 * are formed cumulatively while walking the harmonics of each fundamental cell once,
 *     S_{H_l}[k][c] = S_{H_{l-1}}[k][c] + sum_{h = H_{l-1}+1}^{H_l} P[row(h z_k)][h c],
 * and level l's cells with S_{H_l} > thresholds[l] go to level l's own list.  Each level's candidates are exactly
 * (same cells, same float32 sums bit for bit) those of fdas_harmonic_sum_threshold(nharm[l], thresholds[l]); the
 * fundamental rows are read once instead of once per H.  One launch on `stream`, no allocation, no host sync.
 *   nharm, thresholds : HOST arrays of nlevels entries, 1 <= nlevels <= 4, nharm strictly increasing, >= 1.
 *   d_cands  : device, nlevels x capacity fdas_candidate, 16-byte aligned; level l's list starts at l * capacity
 *              (not checked when capacity is 0).
 *   d_counts : device, nlevels x uint64, zeroed on `stream` first; counts[l] may exceed capacity (then only the
 *              first `capacity` candidates of that level were stored).  Order within a list is unspecified.
 * Errors: as fdas_harmonic_sum_threshold, plus FDAS_ERR_INVALID_ARG for a bad level list.
 */
fdas_status fdas_harmonic_sums_threshold(fdas_plan *plan, void *stream, const float *d_plane, int32_t nlevels,
                                         const int32_t *nharm, const float *thresholds, fdas_candidate *d_cands,
                                         int64_t capacity, uint64_t *d_counts);

/* Free the plan and everything it owns.  fdas_destroy(NULL) is a no-op returning FDAS_OK. */
fdas_status fdas_destroy(fdas_plan *plan);

/* ---- the real-to-complex transform in front of the correlations ---- */

typedef struct fdas_r2c_plan fdas_r2c_plan; /* opaque; created/destroyed by the library */

/*
 * Plan the transform of a REAL time series of `nsamples` float32 samples into the nsamples/2 complex64 bins the
 * correlations take (PAPER.md:79 Fig. 2, :105 "cuFFT R2C", :190, :219; eq. 5; reading R17):
 *     X[k] = scale * sum_j x[j] exp(-2 pi i j k / nsamples),  k = 0 .. nsamples/2 - 1
 * (DC kept, the Nyquist bin dropped).  nsamples must be a power of two, 2^10 <= nsamples <= 2^25
 * (FDAS_ERR_UNSUPPORTED otherwise).  Allocates two work arrays of nsamples/2 complex64 each and the twiddle tables
 * on the current device and fills the tables (synchronises once).
 */
fdas_status fdas_r2c_plan_create(fdas_r2c_plan **out, int64_t nsamples);

/*
 * Transform one series: four launches on `stream` (three transform passes, untangle), no host
 * synchronisation, no allocation.
 *   d_timeseries : device, nsamples float32, 8-byte aligned; read only.
 *   d_spectrum   : device, nsamples/2 x {float re, float im}, 16-byte aligned; every bin is written.  It can be
 *                  handed to fdas_execute of a plan with nbins = nsamples/2 on the same stream.
 *   scale        : multiplies every bin (1/nsamples-type normalisations are the caller's choice; the paper's
 *                  pipeline normalises the spectrum outside the part it covers).
 * One plan, one stream at a time: the plan's two work arrays are shared by all of its calls, so two calls on the
 * same plan that can overlap on the GPU (different streams with no event between them) race silently.  Calls on
 * one stream, or on separate plans, are safe.  Errors: FDAS_ERR_INVALID_ARG (null pointers, another device
 * current than the plan's), FDAS_ERR_ALIGNMENT, FDAS_ERR_CUDA.
 */
fdas_status fdas_r2c_execute(fdas_r2c_plan *plan, void *stream, const float *d_timeseries, void *d_spectrum,
                             float scale);

/* Free the plan.  fdas_r2c_destroy(NULL) is a no-op returning FDAS_OK. */
fdas_status fdas_r2c_destroy(fdas_r2c_plan *plan);

/*
 * The same transform for callers that may not allocate device memory.
 *
 * Who needs it: a host that cannot call cudaMalloc while it runs.  Examples are an acquisition back-end that split
 * the card's memory once at start-up and must keep the allocator's device-wide lock, its implicit synchronisation
 * and its possible failure (a neighbouring process filled the card) out of its real-time loop, and a plug-in inside
 * a framework whose own memory pool already owns nearly all of the GPU, where an allocation made behind the
 * framework's back fails or starves the framework.  Such a caller cannot use fdas_r2c_plan_create, which allocates.
 *
 * This call needs no plan and calls no cudaMalloc, cudaFree or allocating library routine, on its first call or any
 * later one.  The work arrays and twiddle tables of the transform live in one array that is part of the library's
 * device image: FDAS_R2C_STATIC_BYTES (8.04 MiB) on EVERY GPU that loads libfdas.so, held until the process exits
 * whether or not this call is ever made.  That fixes the limit: nsamples must be a power of two with
 * 2^10 <= nsamples <= FDAS_R2C_STATIC_MAX_SAMPLES (2^20); anything else returns FDAS_ERR_UNSUPPORTED, with the
 * reason in fdas_last_error(NULL).  Longer series need fdas_r2c_plan_create.
 *
 *   stream, d_timeseries, d_spectrum, scale : as for fdas_r2c_execute (caller-owned input and output, nsamples
 *                  float32 in, nsamples/2 complex64 out, 8- and 16-byte aligned, FDAS_ERR_ALIGNMENT otherwise).
 *   result       : the same kernels with the same arguments as fdas_r2c_execute, so the same bits.
 *
 * First call on a device: looks up the array's address on the current device and raises the shared-memory limit of
 * the transform kernels (host-side driver calls, no allocation).  Make that first call per device during start-up,
 * before any stream capture begins.  A call whose nsamples differs from the previous call's on that device first
 * refills the twiddle tables with five small launches on `stream`; otherwise it is the four launches of
 * fdas_r2c_execute.  No host synchronisation.
 *
 * Sharing: all calls on a device use the one array, and it keeps whatever the last call left in it.  Nothing in
 * it has to start at zero (every pass overwrites all it later reads), so back-to-back calls of any sizes on ONE
 * stream are safe.  Two calls that can overlap on the GPU (different streams without an event between them,
 * different host threads on different streams) race on the work arrays and tables and give wrong spectra silently;
 * order them yourself.  Host-side the call is thread-safe (one mutex).
 */
#define FDAS_R2C_STATIC_MAX_SAMPLES (1ll << 20)
#define FDAS_R2C_STATIC_BYTES (8ll * (FDAS_R2C_STATIC_MAX_SAMPLES + 3 * 256 + 4096 + FDAS_R2C_STATIC_MAX_SAMPLES / 4096))
fdas_status fdas_r2c_execute_static(void *stream, const float *d_timeseries, int64_t nsamples, void *d_spectrum,
                                    float scale);

/* ---- red-noise removal and block normalisation between the transform and the correlations (8(f) F3) ---- */

typedef enum { FDAS_WHITEN_MEDIAN = 0, FDAS_WHITEN_MEAN = 1 } fdas_whiten_statistic;

/*
 * Scale every block of `block` consecutive bins of a spectrum by one positive real number taken from the block's own
 * Fourier powers (Fig. 2; the paper names the two steps without formulas -- DESIGN.md readings R19, R20):
 *     out[j] = A[j] / sqrt(stat_b),  b = j / block  (blocks start at bin 0; the last one may be shorter)
 *   FDAS_WHITEN_MEDIAN  stat_b = median |A|^2 / ln 2 : "low frequency (red) noise is removed with the use of a local
 *                       median filter" -- the median is blind to the few bins a signal occupies, and exponentially
 *                       distributed noise powers have median = mean x ln 2, so the noise comes out at unit mean power.
 *                       The median is exact (mean of the two middle values for an even count).
 *   FDAS_WHITEN_MEAN    stat_b = mean |A|^2 : "a short step of normalization on the data of each block" -- call it
 *                       with block = fdas_info.useful so that blocks are the plan's overlap-save blocks.
 * A block whose statistic is 0 is copied unchanged.  Inputs are assumed finite with |A|^2 below the float32 range.
 *   d_spectrum : device, nbins x {float re, float im}, 8-byte aligned; read only (twice).
 *   d_out      : device, same shape; may be d_spectrum itself (in place); must not overlap it otherwise.
 * One launch on `stream` (one CTA per block), no plan, no allocation, no host synchronisation; chains between
 * fdas_r2c_execute and fdas_execute on one stream.
 * Errors: FDAS_ERR_INVALID_ARG (null pointers, nbins <= 0, unknown statistic), FDAS_ERR_UNSUPPORTED (block outside
 * [32, 8192]; text in fdas_last_error(NULL)), FDAS_ERR_ALIGNMENT, FDAS_ERR_CUDA.
 */
fdas_status fdas_whiten(void *stream, const void *d_spectrum, void *d_out, int64_t nbins, int32_t block,
                        int32_t statistic);

/* ---- introspection for harnesses and tests (not on the hot path) ---- */

fdas_status fdas_plan_info(const fdas_plan *plan, fdas_info *out);

/*
 * Copy template k's taps to the host (synchronises): host_re_im receives
 * 2*(2*halfwidth_k+1) doubles, interleaved (re, im), index d + halfwidth_k <-> tap d.
 * The buffer must hold 2*(2*info.halfwidth+1) doubles.  Needs fdas_make_templates.
 * With interbin = 2, k in [ntemplates, 2*ntemplates) addresses the half-bin bank of template
 * k - ntemplates: index d + halfwidth_k <-> h_z(d - 1/2), d = -halfwidth_k+1..halfwidth_k (index 0 is 0).
 */
fdas_status fdas_get_taps(fdas_plan *plan, int32_t k, double *host_re_im, int32_t *halfwidth_k);

/*
 * Copy template k's spectrum H_k[0..L-1] to the host in NATURAL frequency order
 * (synchronises): host_re_im receives 2*seglen floats (re, im).
 */
fdas_status fdas_get_template_spectrum(fdas_plan *plan, int32_t k, float *host_re_im);

/*
 * Sustained FP32 FMA throughput of the device's plain ALUs (the "alu" roofline
 * denominator): runs `iters` dependent-chain FMA sweeps on every SM, enqueued on `stream`,
 * synchronises, and returns TFLOP/s (2 flops per FMA) in *tflops.
 */
fdas_status fdas_measure_fp32_peak(void *stream, int32_t iters, double *tflops);

/* Number of kernels the library has launched in this process (for bench accounting). */
int64_t fdas_launch_count(void);

const char *fdas_status_string(fdas_status s);
/* Text of the last CUDA error seen by this plan ("" if none); plan = NULL: of the calling thread's last
 * failed fdas_plan_create, fdas_r2c_plan_create, fdas_r2c_execute, fdas_r2c_execute_static or fdas_whiten. */
const char *fdas_last_error(const fdas_plan *plan);

#ifdef __cplusplus
}
#endif
#endif /* FDAS_H_ */
