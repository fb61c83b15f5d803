/*
 * FDAS oracle -- TEST INFRASTRUCTURE ONLY (not the product path).
 *
 * Plain fp64 direct (non-FFT) evaluation of the correlation technique,
 * PAPER.md:65-69 (section 2, eq. 3):
 *
 *     y_z[r] = sum_{d=-m}^{+m}  A[r+d] * conj(h_z[d]),   A[j] := 0 for j<0 or j>=N
 *
 * "correlating the m bins around r0 with the frequency reversed and complex
 * conjugated template".  The overlap-save FFT pipeline of PAPER.md:75-77 is an
 * exact (up to rounding) evaluation of this same sum, so the oracle is the
 * definition written out.  Zero extension at both ends: DESIGN.md reading R7
 * ("initial zero-padding at the beginning of the input array").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference
 * legs may call this.  It shares no code with the CUDA path.
 *
 * Layouts: A is N interleaved (re,im) float32 pairs (the same complex64 values the
 * GPU receives, up-converted to double here); h is 2m+1 interleaved (re,im) doubles,
 * h[d+m] <-> tap d; y is interleaved (re,im) doubles.
 */
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* One output: eq. 3 at column r (r may lie outside [0,N); the sum uses the zero extension). */
static void correlate_one(const float *A, int64_t N, const double *h, int32_t m,
                          int64_t r, double *yre, double *yim)
{
    double sr = 0.0, si = 0.0;
    for (int32_t d = -m; d <= m; ++d) {
        int64_t j = r + d;
        if (j < 0 || j >= N) continue;              /* A[j] := 0 outside the spectrum */
        double ar = (double)A[2 * j], ai = (double)A[2 * j + 1];
        double hr = h[2 * (d + m)], hi = h[2 * (d + m) + 1];
        /* A * conj(h) = (ar + i ai)(hr - i hi) */
        sr += ar * hr + ai * hi;
        si += ai * hr - ar * hi;
    }
    *yre = sr;
    *yim = si;
}

/* y[r] for r = r_begin .. r_begin + r_count - 1 (contiguous columns of one template row). */
void fdas_oracle_correlate(const float *A, int64_t N, const double *h, int32_t m,
                           int64_t r_begin, int64_t r_count, double *y)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < r_count; ++i)
        correlate_one(A, N, h, m, r_begin + i, &y[2 * i], &y[2 * i + 1]);
}

/* y at an arbitrary list of columns (sampled parity checks at full size). */
void fdas_oracle_correlate_at(const float *A, int64_t N, const double *h, int32_t m,
                              const int64_t *cols, int64_t ncols, double *y)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < ncols; ++i)
        correlate_one(A, N, h, m, cols[i], &y[2 * i], &y[2 * i + 1]);
}

/*
 * Discrete Fourier transform of a REAL time series, eq. 5 written out:
 *
 *     X[k] = sum_{j=0}^{n-1} x[j] exp(-2 pi i j k / n)          (unnormalised, forward sign)
 *
 * at the listed bins k (any integers; the sum is the definition, so bins >= n/2 are allowed and give the
 * conjugate-symmetric half).  This is the "long real-to-complex FFT" in front of the correlations
 * (PAPER.md:79 Fig. 2, :105 "cuFFT R2C", :190, :219), evaluated directly: O(n) per bin, the phase
 * reduced exactly in integers (j k mod n) before the one sincos per term.  x: n float32 samples (the values
 * the GPU receives, up-converted); out: interleaved (re, im) doubles.
 */
#include <math.h>
void fdas_oracle_dft_real_at(const float *x, int64_t n, const int64_t *bins, int64_t nb, double *out)
{
    const double w = -2.0 * 3.14159265358979323846264338327950288 / (double)n;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t b = 0; b < nb; ++b) {
        const int64_t k = ((bins[b] % n) + n) % n;
        double sr = 0.0, si = 0.0;
        int64_t ph = 0;                              /* (j k) mod n, advanced by k per sample */
        for (int64_t j = 0; j < n; ++j) {
            const double a = w * (double)ph;
            sr += (double)x[j] * cos(a);
            si += (double)x[j] * sin(a);
            ph += k;
            if (ph >= n) ph -= n;
        }
        out[2 * b] = sr;
        out[2 * b + 1] = si;
    }
}

int32_t fdas_oracle_threads(void)
{
#ifdef _OPENMP
    return (int32_t)omp_get_max_threads();
#else
    return 1;
#endif
}
