// Real-to-complex transform of the time series in front of the correlations.
//
// PAPER.md:79 (Fig. 2: the FDAS pipeline starts from the FFT of the time series), :105 ("cuFFT R2C"), :190 and
// :219 (the long real FFT is inside every timing of the paper), eq. 5:
//
//     X[k] = scale * sum_{j=0}^{n-1} x[j] exp(-2 pi i j k / n),   k = 0 .. n/2 - 1     (reading R17: DC kept,
//                                                                                       Nyquist bin dropped)
// n = 2^p real samples.  The series is read as M = n/2 complex numbers z[j] = x[2j] + i x[2j+1]; Z = DFT_M(z) by a
// three-factor decomposition M = N1 N2 N3 (j = j1 N2 N3 + j2 N3 + j3, k = k1 + N1 k2 + N1 N2 k3; every factor
// <= 256), i.e. the four-step scheme applied twice, three passes through memory plus the untangle:
//
//   pass A  transforms of length N1 over j1 (stride N2 N3), times exp(-2 pi i j' k1 / M), j' = j2 N3 + j3  -> [k1][j']
//   pass B  per k1: transforms of length N2 over j2 (stride N3), times exp(-2 pi i j3 k2 / (N2 N3))         -> [k1][k2][j3]
//   pass C  transforms of length N3 over j3 (contiguous), stored transposed at k = k1 + N1 k2 + N1 N2 k3    -> spectrum
//   pass D  untangle in place: E = (Z[k] + conj Z[M-k]) / 2, O = (Z[k] - conj Z[M-k]) / 2i,
//           X[k] = E + W^k O, X[M-k] = conj(E - W^k O), W = exp(-2 pi i / n)
//
// A CTA holds 2^ltile transforms side by side in shared memory (rows padded to R + 1 elements).  In passes A and
// B the side-by-side transforms are ADJACENT COLUMNS (the innermost, contiguous index), in pass C adjacent k1, so
// every global access of every pass is a run of 2^ltile * 8 contiguous bytes (256 B at ltile = 5); inside the CTA
// lane <-> transform, so butterflies, twiddle reads (one address per warp) and the bit-reversed read-out are free
// of bank conflicts.  The in-CTA transform is an in-place radix-4 decimation in frequency (two fused radix-2
// levels per shared-memory round trip, a last radix-2 level when log2 R is odd); its bit-reversed order is
// undone when the tile is read back out, so no separate re-ordering pass exists (PAPER.md:156-180 uses the same
// property).  All twiddles come from fp64-evaluated tables: exp(-2 pi i j / R) per pass and a two-level table of
// exp(-2 pi i t / n).  Traffic: 4 x (8M read + 8M write) = 32 n bytes against the compulsory 8 n (4 n in, 4 n
// out); up to n = 2^23 the 12 n-byte working set stays in the 126 MB L2 between passes.
#pragma once
#include "fdas_fft.cuh"
#include <stdint.h>

namespace fdas {

struct R2CParams {
    const float2 *in;     // this pass's input
    float2 *out;          // this pass's output
    const float2 *wR;     // exp(-2 pi i j / R), j < R (this pass's transform length)
    const float2 *tlo;    // exp(-2 pi i t / n), t < 4096
    const float2 *thi;    // exp(-2 pi i 4096 t / n), t < ceil(n / 4096)
    long long M;          // n / 2
    long long inner;      // passes A / B: columns per slab (A: N2 N3, B: N3); pass C: N3
    long long slab;       // passes A / B: elements per slab (A: M, B: N2 N3)
    long long tmul;       // passes A / B: twiddle exp(-2 pi i tmul col k / n)  (A: 2, B: 2 N1)
    int N1, N2;           // pass C: output index k1 + N1 k2 + N1 N2 k3
    int log2R;            // log2 of this pass's transform length R
    int ltile;            // log2 of the transforms per CTA
    float scale;
};

#ifdef __CUDACC__

__device__ __forceinline__ float2 r2c_wn(const R2CParams &p, long long t)   // exp(-2 pi i t / n), 0 <= t < n
{
    return cmul(__ldg(p.thi + (t >> 12)), __ldg(p.tlo + (t & 4095)));
}

// In-place DIF of 2^ltile transforms of length R = 2^log2R held in buf[c * RS + i]; output bit-reversed.
// sw: exp(-2 pi i j / R) in shared memory.  All index arithmetic is shifts and masks (R, tile are powers of two).
__device__ __forceinline__ void r2c_fft_tile(float2 *buf, int RS, int ltile, int log2R, const float2 *sw)
{
    const int tmask = (1 << ltile) - 1;
    int ll = log2R;                                       // log2 of the current block length
    for (; ll >= 2; ll -= 2) {
        const int lq = ll - 2, q = 1 << lq, ws = log2R - ll;
        const int nb = 1 << (ltile + log2R - 2);
        for (int e = threadIdx.x; e < nb; e += blockDim.x) {
            const int c = e & tmask, b = e >> ltile;      // lane <-> transform: conflict-free, twiddles broadcast
            const int blk = b >> lq, j = b & (q - 1);
            float2 *a = buf + c * RS + (blk << ll) + j;
            const float2 a0 = a[0], a1 = a[q], a2 = a[2 * q], a3 = a[3 * q];
            const float2 b0 = cadd(a0, a2), b1 = cadd(a1, a3);
            const float2 b2 = cmul(csub(a0, a2), sw[j << ws]);
            const float2 b3 = cmul(csub(a1, a3), sw[(j + q) << ws]);
            const float2 w2 = sw[(2 * j) << ws];
            a[0] = cadd(b0, b1);
            a[q] = cmul(csub(b0, b1), w2);
            a[2 * q] = cadd(b2, b3);
            a[3 * q] = cmul(csub(b2, b3), w2);
        }
        __syncthreads();
    }
    if (ll == 1) {
        const int nb = 1 << (ltile + log2R - 1);
        for (int e = threadIdx.x; e < nb; e += blockDim.x) {
            const int c = e & tmask, b = e >> ltile;
            float2 *a = buf + c * RS + 2 * b;
            const float2 a0 = a[0], a1 = a[1];
            a[0] = cadd(a0, a1);
            a[1] = csub(a0, a1);
        }
        __syncthreads();
    }
}

// passes A and B: transforms over a strided index for 2^ltile adjacent columns.  grid = (inner >> ltile, slabs)
__global__ void __launch_bounds__(512) r2c_cols_kernel(const R2CParams p)
{
    extern __shared__ __align__(16) unsigned char r2c_smem[];
    float2 *buf = reinterpret_cast<float2 *>(r2c_smem);
    const int R = 1 << p.log2R, RS = R + 1, lt = p.ltile, tile = 1 << lt;
    float2 *sw = buf + tile * RS;
    const long long col0 = (long long)blockIdx.x << lt;
    const float2 *in = p.in + (long long)blockIdx.y * p.slab;
    float2 *out = p.out + (long long)blockIdx.y * p.slab;
    for (int e = threadIdx.x; e < R; e += blockDim.x) sw[e] = __ldg(p.wR + e);
    for (int e = threadIdx.x; e < (R << lt); e += blockDim.x) {
        const int c = e & (tile - 1), j = e >> lt;
        buf[c * RS + j] = __ldg(in + (long long)j * p.inner + col0 + c);
    }
    __syncthreads();
    r2c_fft_tile(buf, RS, lt, p.log2R, sw);
    const int sh = 32 - p.log2R;
    for (int e = threadIdx.x; e < (R << lt); e += blockDim.x) {
        const int c = e & (tile - 1), k = e >> lt;
        const float2 v = buf[c * RS + (int)(__brev((unsigned)k) >> sh)];
        out[(long long)k * p.inner + col0 + c] = cmul(v, r2c_wn(p, p.tmul * (col0 + c) * k));
    }
}

// pass C: transforms over the contiguous index j3 of the rows (k1, k2), 2^ltile adjacent k1 per CTA.
// grid = (N1 >> ltile, N2)
__global__ void __launch_bounds__(512) r2c_rows_kernel(const R2CParams p)
{
    extern __shared__ __align__(16) unsigned char r2c_smem[];
    float2 *buf = reinterpret_cast<float2 *>(r2c_smem);
    const int R = 1 << p.log2R, RS = R + 1, lt = p.ltile, tile = 1 << lt;
    float2 *sw = buf + tile * RS;
    const long long k1_0 = (long long)blockIdx.x << lt, k2 = blockIdx.y;
    for (int e = threadIdx.x; e < R; e += blockDim.x) sw[e] = __ldg(p.wR + e);
    for (int e = threadIdx.x; e < (R << lt); e += blockDim.x) {
        const int c = e >> p.log2R, j3 = e & (R - 1);
        buf[c * RS + j3] = __ldg(p.in + ((k1_0 + c) * p.N2 + k2) * R + j3);
    }
    __syncthreads();
    r2c_fft_tile(buf, RS, lt, p.log2R, sw);
    const int sh = 32 - p.log2R;
    for (int e = threadIdx.x; e < (R << lt); e += blockDim.x) {
        const int c = e & (tile - 1), k3 = e >> lt;
        p.out[k1_0 + c + (long long)p.N1 * (k2 + (long long)p.N2 * k3)] = buf[c * RS + (int)(__brev((unsigned)k3) >> sh)];
    }
}

// pass D: Z -> X in place, one thread per pair (k, M - k), k = 0 .. M/2
__global__ void __launch_bounds__(256) r2c_untangle_kernel(const R2CParams p)
{
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k > p.M / 2) return;
    float2 *z = p.out;
    if (k == 0) {
        const float2 a = z[0];
        z[0] = make_float2(p.scale * (a.x + a.y), 0.f);       // DC; the Nyquist bin a.x - a.y is dropped (R17)
        return;
    }
    const float2 a = z[k], b = z[p.M - k];
    const float2 e = make_float2(0.5f * (a.x + b.x), 0.5f * (a.y - b.y));     // (a + conj b) / 2
    const float2 o = make_float2(0.5f * (a.y + b.y), -0.5f * (a.x - b.x));    // (a - conj b) / 2i
    const float2 wo = cmul(o, r2c_wn(p, k));
    z[k] = make_float2(p.scale * (e.x + wo.x), p.scale * (e.y + wo.y));
    if (k != p.M - k) z[p.M - k] = make_float2(p.scale * (e.x - wo.x), -p.scale * (e.y - wo.y));
}

// exp(-2 pi i j step / len) for j < count, fp64-evaluated
__global__ void r2c_table_kernel(float2 *tab, long long count, long long step, long long len)
{
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= count) return;
    const long long t = (j * step) % len;
    double s, c;
    sincospi(-2.0 * (double)t / (double)len, &s, &c);
    tab[j] = make_float2((float)c, (float)s);
}

#endif // __CUDACC__

} // namespace fdas
