// Plan-time template generation on the device (fp64).
//
//  a0  taps: h_z(d) = int_0^1 exp(2 pi i [ -d u + z (u^2 - u)/2 ]) du -- the "predicted
//      normalised Fourier response" to a constant frequency derivative (formula
//      not printed there, reading R1), evaluated from its Fresnel-integral closed form
//          z > 0, q = -d - z/2, Y = q sqrt(2/z), Z = (q+z) sqrt(2/z):
//          h_z(d) = exp(-i pi q^2 / z) / sqrt(2 z) * { [C(Z)-C(Y)] + i [S(Z)-S(Y)] }
//          z < 0: h_z(d) = conj(h_{-z}(-d));   z = 0: Kronecker delta at integer d.
//      Bank 1 (2-bin Fourier interpolation, reading R16) holds the same response
//      at the half-integer offsets d - 1/2, d = -m_z+1..m_z (z = 0: exp(-i pi x) sin(pi x)/(pi x)).
//  a1  spectra: H_z[f] = (1/L) sum_d conj(h_z[d]) exp(+2 pi i d f / L)   (the
//      filter centred at bin 0, halves at both ends of the L-array; 1/L of eq. 6 folded in, R6),
//      written in the register order of the fused kernel's un-permuted FFT.
#pragma once
#include "fdas_kernel.cuh"
#include "fdas_kernel8k.cuh"
#include "fdas_kernel2.cuh"
#include "fdas_kernel3.cuh"
#include "fdas_r2c.cuh"
#include "fdas_whiten.cuh"

namespace fdas {

// Fresnel integrals C(x) = int_0^x cos(pi t^2/2) dt, S(x) = int_0^x sin(pi t^2/2) dt, fp64.
//   |x| < 1.8 : Maclaurin series (terms stay below ~200, so cancellation costs < 3 digits)
//   else      : C + iS = (1+i)/2 * (1 - erfc(w)), w = (sqrt(pi)/2)(1-i)x, with erfc from its
//               continued fraction  exp(-w^2)/sqrt(pi) * 1/(w + (1/2)/(w + 1/(w + (3/2)/(w + ...))))
//               evaluated bottom-up with a fixed depth (80 levels reach 1e-16 at |x| = 1.8).
__device__ inline void fresnel_cs(double x, double &C, double &S)
{
    const double ax = fabs(x);
    double c, s;
    if (ax < 1.8) {
        const double a = 1.5707963267948966192313216916398 * ax * ax; // pi/2 x^2
        double term = ax;                                              // a^k x / k!, k = 0
        c = 0.0;
        s = 0.0;
        for (int n = 0; n < 32; ++n) {
            const double sg = (n & 1) ? -1.0 : 1.0;
            c += sg * term / (4 * n + 1);
            term *= a / (2 * n + 1);
            s += sg * term / (4 * n + 3);
            term *= a / (2 * n + 2);
        }
    } else {
        const double k = 0.88622692545275801364908374167057 * ax; // sqrt(pi)/2 * x
        const double wr = k, wi = -k;                              // w = k (1 - i)
        double fr = wr, fi = wi;
        const int depth = ax > 6.0 ? 24 : (ax > 3.0 ? 48 : 96);
        for (int j = depth; j >= 1; --j) {
            const double g = 0.5 * j / (fr * fr + fi * fi);        // (j/2) / f = (j/2) conj(f)/|f|^2
            const double nr = wr + g * fr, ni = wi - g * fi;
            fr = nr;
            fi = ni;
        }
        // erfc(w) = exp(-w^2)/(sqrt(pi) f), exp(-w^2) = exp(+i pi x^2 / 2)
        double es, ec;
        sincospi(0.5 * ax * ax, &es, &ec);
        const double inv = 0.56418958354775628694807945156077 / (fr * fr + fi * fi); // 1/sqrt(pi)/|f|^2
        const double er = inv * (ec * fr + es * fi), ei = inv * (es * fr - ec * fi); // e^{..} conj(f)
        // (1+i)/2 * (1 - erfc)
        const double ur = 1.0 - er, ui = -ei;
        c = 0.5 * (ur - ui);
        s = 0.5 * (ur + ui);
    }
    C = x < 0 ? -c : c;
    S = x < 0 ? -s : s;
}

// closed form for z > 0
__device__ inline double2 response_closed_form(double z, double d)
{
    const double q = -d - 0.5 * z;
    const double sc = sqrt(2.0 / z);
    double CY, SY, CZ, SZ;
    fresnel_cs(q * sc, CY, SY);
    fresnel_cs((q + z) * sc, CZ, SZ);
    double ps, pc;
    sincospi(-q * q / z, &ps, &pc);
    const double a = CZ - CY, b = SZ - SY, n = 1.0 / sqrt(2.0 * z);
    return make_double2(n * (pc * a - ps * b), n * (pc * b + ps * a));
}

__device__ inline int tap_halfwidth(double z)
{
    return (int)ceil(fabs(z) * 0.5 - 1e-12) + 16; // R4: ceil(|z|/2) + 16
}

// taps[k][d + m], d = -m..m (m = bank half-width); zero for |d| > m_z.  half = 1: bank 1, the tap at
// index d is h_z(d - 1/2), d = -m_z+1..m_z.
__global__ void make_taps_kernel(double2 *taps, int K, int m, double zmax, double dz, int half)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    const int w = 2 * m + 1;
    if (idx >= K * w) return;
    const int k = idx / w, d = idx % w - m;
    const int center = (K - 1) / 2;
    const double z = (k == center) ? 0.0 : -zmax + k * dz;
    const int mz = tap_halfwidth(z);
    double2 h = make_double2(0.0, 0.0);
    if (d >= -mz + half && d <= mz) {
        const double x = (double)d - 0.5 * half;
        if (z == 0.0) {
            if (half) {                                  // exp(-i pi x) sinc(x) at half-integer x
                double sn, cs;
                sincospi(x, &sn, &cs);
                const double sc = sn / (3.14159265358979323846264338327950288 * x);
                h = make_double2(cs * sc, -sn * sc);
            } else {
                h.x = (d == 0) ? 1.0 : 0.0;
            }
        } else if (z > 0.0) {
            h = response_closed_form(z, x);
        } else {
            h = response_closed_form(-z, -x);
            h.y = -h.y;
        }
    }
    taps[idx] = h;
}

__global__ void make_wtab_kernel(float2 *wtab, int L)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= L) return;
    double s, c;
    sincospi(-2.0 * j / L, &s, &c);
    wtab[j] = make_float2((float)c, (float)s);
}

// hperm[pair][i/2][tid] (float4 = two complex) for the rows z <= 0 (pair = row index k).
// nbanks = 2: slot = pair * 2 + bank; `taps` points at the bank's tap array.
// MAP = 3: register order of fdas_kernel3.cuh (freq_to_reg3), else of fdas_kernel.cuh.
template <int L, int MAP = 0>
__global__ void make_spectra_kernel(float2 *hperm, const double2 *taps, int npairs, int m,
                                    double zmax, double dz, int K, int nbanks, int bank)
{
    using G = Geo<L>;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= npairs * L) return;
    const int pair = idx / L, f = idx % L;
    const int center = (K - 1) / 2;
    const double z = (pair == center) ? 0.0 : -zmax + pair * dz;
    const int mz = tap_halfwidth(z);
    const double2 *h = taps + (size_t)pair * (2 * m + 1) + m;
    double sr = 0.0, si = 0.0;
    for (int d = -mz; d <= mz; ++d) {
        int r = (int)(((long long)d * f) % L);
        if (r < 0) r += L;
        double s, c;
        sincospi(2.0 * r / L, &s, &c);           // exp(+2 pi i d f / L)
        const double2 t = h[d];
        sr += t.x * c + t.y * s;                  // conj(h) * e
        si += t.x * s - t.y * c;
    }
    int tid, i;
    if constexpr (MAP == 3) freq_to_reg3<L>(f, tid, i);
    else freq_to_reg<L>(f, tid, i);
    const size_t off = ((((size_t)pair * nbanks + bank) * (G::PTS / 2) + (i >> 1)) * G::T + tid) * 2 + (i & 1);
    hperm[off] = make_float2((float)(sr / L), (float)(si / L));
}

// seglen 8192: hperm[pair][half][i/2][tid] with half 0 = H[k], half 1 = H[k + 4096], k < 4096 in
// the slot order of Geo<4096> (fdas_kernel8k.cuh).
__global__ void make_spectra_kernel_8k(float2 *hperm, const double2 *taps, int npairs, int m,
                                       double zmax, double dz, int K, int nbanks, int bank)
{
    using G = Geo<4096>;
    constexpr int L = 8192;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= npairs * L) return;
    const int pair = idx / L, f = idx % L;
    const int center = (K - 1) / 2;
    const double z = (pair == center) ? 0.0 : -zmax + pair * dz;
    const int mz = tap_halfwidth(z);
    const double2 *h = taps + (size_t)pair * (2 * m + 1) + m;
    double sr = 0.0, si = 0.0;
    for (int d = -mz; d <= mz; ++d) {
        int r = (int)(((long long)d * f) % L);
        if (r < 0) r += L;
        double s, c;
        sincospi(2.0 * r / L, &s, &c);
        const double2 t = h[d];
        sr += t.x * c + t.y * s;
        si += t.x * s - t.y * c;
    }
    int tid, i;
    freq_to_reg<4096>(f & 4095, tid, i);
    const int half = f >> 12;
    const size_t off = (((((size_t)pair * nbanks + bank) * 2 + half) * (G::PTS / 2) + (i >> 1)) * G::T + tid) * 2 + (i & 1);
    hperm[off] = make_float2((float)(sr / L), (float)(si / L));
}

// FP32 FMA throughput probe: 8 independent chains per thread.
__global__ void fp32_peak_kernel(float *out, int iters, float a, float b)
{
    float v0 = threadIdx.x, v1 = v0 + 1, v2 = v0 + 2, v3 = v0 + 3, v4 = v0 + 4, v5 = v0 + 5,
          v6 = v0 + 6, v7 = v0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            v0 = fmaf(v0, a, b); v1 = fmaf(v1, a, b); v2 = fmaf(v2, a, b); v3 = fmaf(v3, a, b);
            v4 = fmaf(v4, a, b); v5 = fmaf(v5, a, b); v6 = fmaf(v6, a, b); v7 = fmaf(v7, a, b);
        }
    }
    const float s = v0 + v1 + v2 + v3 + v4 + v5 + v6 + v7;
    if (s == 12345.678f) out[0] = s;
}

// Harmonic summing of a stored plane + threshold (fdas_harmonic_sum_threshold, include/fdas.h; PAPER.md:73, :79,
// :331; reading R18): S = sum_h P[row(h z_k)][h c] for the fundamental column c of row blockIdx.x / nbx (column
// block blockIdx.x % nbx; rows are folded into x because gridDim.y stops at 65 535).  A thread forms
// four sums (columns c0 + {0, 1, 2, 3} * blockDim.x, so that every load of a warp is a run of consecutive addresses
// with stride h) to keep 4 H independent loads in flight; the order of the additions is h = 1, 2, .. H.
__global__ void __launch_bounds__(256) harmonic_sum_kernel(const float *__restrict__ plane, long long ncols, int K,
                                                           int nharm, int row_first, unsigned nbx, float threshold,
                                                           Candidate *cands, long long capacity,
                                                           unsigned long long *count)
{
    const long long nc = (ncols - 1) / nharm + 1;
    const unsigned by = blockIdx.x / nbx, bx = blockIdx.x - by * nbx;
    const long long c0 = (long long)bx * (4 * blockDim.x) + threadIdx.x;
    const int k = row_first + (int)by, center = (K - 1) / 2;
    float s[4] = {0.f, 0.f, 0.f, 0.f};
    for (int h = 1; h <= nharm; ++h) {
        const float *row = plane + (size_t)(center + h * (k - center)) * ncols;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const long long c = c0 + (long long)j * blockDim.x;
            if (c < nc) s[j] += __ldg(row + h * c);
        }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const long long c = c0 + (long long)j * blockDim.x;
        if (c < nc && s[j] > threshold) {
            const unsigned long long slot = atomicAdd(count, 1ull);
            if (slot < (unsigned long long)capacity) {
                Candidate cd;
                cd.col = c;
                cd.row = k;
                cd.power = s[j];
                cands[slot] = cd;
            }
        }
    }
}

// Harmonic sums for several H in ONE walk over the harmonics of a fundamental cell (fdas_harmonic_sums_threshold,
// include/fdas.h; reading R18): S_{H_l} = S_{H_{l-1}} + sum_{h = H_{l-1}+1}^{H_l} P[row(h z_k)][h c],
// compared with level l's threshold as soon as it is complete and appended to level l's own list.  The grid covers the
// rows and columns of the first level; a cell leaves the walk at the first level whose domain (|z_k| <= zmax / H_l,
// H_l c <= ncols - 1) it is outside -- for a whole CTA when its row or its column block is (uniform branch).  The
// additions run in the order h = 1, 2, .. like harmonic_sum_kernel's, so each level's sums are bit-identical to a
// separate launch of that kernel; the fundamental rows are read once instead of once per H.
struct HarmonicLevels {
    int nlevels;
    int nharm[4];
    float threshold[4];
    long long capacity;          // per level
    Candidate *cands;            // nlevels x capacity
    unsigned long long *counts;  // nlevels
};

__global__ void __launch_bounds__(256) harmonic_sums_kernel(const float *__restrict__ plane, long long ncols, int K,
                                                            unsigned nbx, const HarmonicLevels lv)
{
    const unsigned by = blockIdx.x / nbx, bx = blockIdx.x - by * nbx;
    const int center = (K - 1) / 2;
    const int dk = (int)by - center / lv.nharm[0];                 // row offset from z = 0 of this CTA's fundamental
    const long long cb = (long long)bx * (4 * blockDim.x), c0 = cb + threadIdx.x;
    float s[4] = {0.f, 0.f, 0.f, 0.f};
    int h = 1;
#pragma unroll
    for (int l = 0; l < 4; ++l) {                                  // unrolled: lv stays in the parameter bank
        if (l >= lv.nlevels) return;
        const int hl = lv.nharm[l];
        const long long nc = (ncols - 1) / hl + 1;
        if ((dk < 0 ? -dk : dk) > center / hl || cb >= nc) return;
        for (; h <= hl; ++h) {
            const float *row = plane + (size_t)(center + h * dk) * ncols;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const long long c = c0 + (long long)j * blockDim.x;
                if (c < nc) s[j] += __ldg(row + h * c);
            }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const long long c = c0 + (long long)j * blockDim.x;
            if (c < nc && s[j] > lv.threshold[l]) {
                const unsigned long long slot = atomicAdd(lv.counts + l, 1ull);
                if (slot < (unsigned long long)lv.capacity) {
                    Candidate cd;
                    cd.col = c;
                    cd.row = center + dk;
                    cd.power = s[j];
                    lv.cands[(size_t)l * lv.capacity + slot] = cd;
                }
            }
        }
    }
}

} // namespace fdas
