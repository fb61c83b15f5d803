// Register-resident radix-2^k DFT butterflies for the fused FDAS kernel.
//
// PAPER.md:133-139 (eqs. 5, 6): forward DFT uses exp(-2 pi i nm/N), inverse exp(+2 pi i nm/N),
// both unnormalised.  PAPER.md:156-180: the forward transform is decimation-in-frequency, the
// inverse decimation-in-time, so no re-ordering pass is needed (the pointwise product does not
// care about element order).  Here each pass is a radix-4/8/16/32 DFT held entirely in
// registers (natural order in, natural order out; the re-ordering inside a pass is register
// renaming and costs nothing); the inter-pass transposes live in the kernel.
//
// DIR = -1: forward (eq. 5), DIR = +1: inverse (eq. 6).
#pragma once
#include <cuda_runtime.h>

#define FDAS_HD __host__ __device__ __forceinline__

namespace fdas {

// cos(2 pi k / 32), k = 0..8 (fp64 literals rounded to fp32 at compile time)
FDAS_HD constexpr float cos32(int k)
{
    return k == 0 ? 1.0f
         : k == 1 ? 0.98078528040323044912618223613424f
         : k == 2 ? 0.92387953251128675612818318939679f
         : k == 3 ? 0.83146961230254523707878837761791f
         : k == 4 ? 0.70710678118654752440084436210485f
         : k == 5 ? 0.55557023301960222474283081394853f
         : k == 6 ? 0.38268343236508977172845998403040f
         : k == 7 ? 0.19509032201612826784828486847702f
         : 0.0f;
}
// cos / sin of 2 pi idx / 32 for idx in [0, 16]
FDAS_HD constexpr float cosw(int idx) { return idx <= 8 ? cos32(idx) : -cos32(16 - idx); }
FDAS_HD constexpr float sinw(int idx) { return idx <= 8 ? cos32(8 - idx) : cos32(idx - 8); }

FDAS_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
FDAS_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
FDAS_HD float2 cmul(float2 a, float2 w)
{
    return make_float2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x);
}
FDAS_HD float2 cmul_conj(float2 a, float2 w) // a * conj(w)
{
    return make_float2(a.x * w.x + a.y * w.y, a.y * w.x - a.x * w.y);
}

// tan(2 pi k / 32), k = 0..4 (|tan| <= 1), for the 6-FMA twiddled butterfly below
FDAS_HD constexpr float tan32(int k)
{
    return k == 0 ? 0.0f
         : k == 1 ? 0.19891236737965800691159762264468f
         : k == 2 ? 0.41421356237309504880168872420970f
         : k == 3 ? 0.66817863791929891999775768652308f
         : 1.0f;
}

// One radix-2 DIT butterfly with the compile-time twiddle w = exp(DIR * 2 pi i * J / LEN):
//   e' = e + w o,  o' = e - w o.     J in [0, LEN/2), LEN in {2,4,8,16,32}
// Non-trivial twiddles use the 6-FMA form: w o = s * (u, v) with (u, v) = o rotated by a
// unit-free factor (1, t) or (t, 1), |t| = tan <= 1, so that e +- s*(u,v) are 4 FMAs.
template <int DIR, int J, int LEN>
FDAS_HD void bfly(float2 &e, float2 &o)
{
    constexpr int idx = J * (32 / LEN); // angle = DIR * 2 pi idx / 32, idx in [0,16)
    const float2 ee = e;
    if constexpr (idx == 0) {
        e = cadd(ee, o);
        o = csub(ee, o);
    } else if constexpr (idx == 8) { // w = DIR * i
        const float2 t = (DIR > 0) ? make_float2(-o.y, o.x) : make_float2(o.y, -o.x);
        e = cadd(ee, t);
        o = csub(ee, t);
    } else {
        // w = c + i s with c = cos(a), s = DIR*sin(a), a = 2 pi idx/32 in (0, pi), a != pi/2.
        // Write w = g * (p + i q) with (p, q) = (1, tan) when |c| >= |s|, else (cot, 1); g = c or s.
        constexpr int r = idx <= 8 ? idx : 16 - idx;           // reflect to [0, 8]
        constexpr bool cos_major = r <= 4;                       // |cos| >= |sin|
        constexpr float tt = cos_major ? tan32(r) : tan32(8 - r); // |sin/cos| or |cos/sin|
        constexpr float cs = idx <= 8 ? 1.0f : -1.0f;            // sign of cos
        constexpr float sn = DIR > 0 ? 1.0f : -1.0f;             // sign of sin
        float u, v, g;
        if constexpr (cos_major) {
            // w = c (1 + i q), q = s/c
            constexpr float q = sn * cs * tt;
            g = cosw(idx);
            u = fmaf(-q, o.y, o.x);
            v = fmaf(q, o.x, o.y);
        } else {
            // w = s (p + i), p = c/s
            constexpr float pq = sn * cs * tt;
            g = sn * sinw(idx);
            u = fmaf(pq, o.x, -o.y);
            v = fmaf(pq, o.y, o.x);
        }
        e = make_float2(fmaf(g, u, ee.x), fmaf(g, v, ee.y));
        o = make_float2(fmaf(-g, u, ee.x), fmaf(-g, v, ee.y));
    }
}


#ifdef __CUDACC__
// ------------------------------------------------------------------ packed (+z, -z) pairs
// The +z and -z transforms of one template slot go through identical
// butterflies, so they are carried as ONE stream of sm_100 packed-fp32 instructions
// (FADD2 / FMUL2 / FFMA2: two fp32 lanes per 64-bit register pair, scalar operands broadcast):
//   re = (Re p, Re q),  im = (Im p, Im q)   with p the z <= 0 transform, q its z >= 0 partner.
// Same FP32-lane throughput as scalar code, half the issue slots.
struct cpk {
    float2 re, im;
};
__device__ __forceinline__ float2 bc2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, neg2(b)); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }

// (p, q) * w for a per-thread twiddle w (the same for both transforms)
__device__ __forceinline__ cpk cmul(cpk a, float2 w)
{
    cpk r;
    r.re = fma2(a.im, bc2(-w.y), mul2(a.re, bc2(w.x)));
    r.im = fma2(a.im, bc2(w.x), mul2(a.re, bc2(w.y)));
    return r;
}

template <int DIR, int J, int LEN>
__device__ __forceinline__ void bfly(cpk &e, cpk &o)
{
    constexpr int idx = J * (32 / LEN);
    const cpk ee = e;
    if constexpr (idx == 0) {
        e.re = add2(ee.re, o.re);
        e.im = add2(ee.im, o.im);
        o.re = sub2(ee.re, o.re);
        o.im = sub2(ee.im, o.im);
    } else if constexpr (idx == 8) { // w = DIR * i:  w o = DIR * (-o.im, o.re)
        const cpk oo = o;
        if constexpr (DIR > 0) {
            e.re = sub2(ee.re, oo.im);
            e.im = add2(ee.im, oo.re);
            o.re = add2(ee.re, oo.im);
            o.im = sub2(ee.im, oo.re);
        } else {
            e.re = add2(ee.re, oo.im);
            e.im = sub2(ee.im, oo.re);
            o.re = sub2(ee.re, oo.im);
            o.im = add2(ee.im, oo.re);
        }
    } else { // 6-FMA twiddled butterfly, see the scalar version above
        constexpr int r = idx <= 8 ? idx : 16 - idx;
        constexpr bool cos_major = r <= 4;
        constexpr float tt = cos_major ? tan32(r) : tan32(8 - r);
        constexpr float cs = idx <= 8 ? 1.0f : -1.0f;
        constexpr float sn = DIR > 0 ? 1.0f : -1.0f;
        float2 u, v;
        float g;
        if constexpr (cos_major) {
            constexpr float q = sn * cs * tt;
            g = cosw(idx);
            u = fma2(bc2(-q), o.im, o.re);
            v = fma2(bc2(q), o.re, o.im);
        } else {
            constexpr float pq = sn * cs * tt;
            g = sn * sinw(idx);
            u = fma2(bc2(pq), o.re, neg2(o.im));
            v = fma2(bc2(pq), o.im, o.re);
        }
        e.re = fma2(bc2(g), u, ee.re);
        e.im = fma2(bc2(g), v, ee.im);
        o.re = fma2(bc2(-g), u, ee.re);
        o.im = fma2(bc2(-g), v, ee.im);
    }
}
#endif // __CUDACC__

template <int R>
FDAS_HD constexpr int bitrev(int i)
{
    int r = 0;
    for (int b = 1; b < R; b <<= 1) {
        r = (r << 1) | (i & 1);
        i >>= 1;
    }
    return r;
}

template <int DIR, int LEN, int G, int J, int R, typename C>
FDAS_HD void dft_level_j(C (&b)[R])
{
    if constexpr (J < LEN / 2) {
        bfly<DIR, J, LEN>(b[G + J], b[G + J + LEN / 2]);
        dft_level_j<DIR, LEN, G, J + 1, R>(b);
    }
}
template <int DIR, int LEN, int G, int R, typename C>
FDAS_HD void dft_level_g(C (&b)[R])
{
    if constexpr (G < R) {
        dft_level_j<DIR, LEN, G, 0, R>(b);
        dft_level_g<DIR, LEN, G + LEN, R>(b);
    }
}
template <int DIR, int LEN, int R, typename C>
FDAS_HD void dft_levels(C (&b)[R])
{
    if constexpr (LEN <= R) {
        dft_level_g<DIR, LEN, 0, R>(b);
        dft_levels<DIR, LEN * 2, R>(b);
    }
}

// In-register DFT of length R (power of two, <= 32): a[k] <- sum_n a[n] exp(DIR 2 pi i n k / R).
template <int DIR, int R, typename C>
FDAS_HD void dft(C (&a)[R])
{
    static_assert(R == 1 || R == 2 || R == 4 || R == 8 || R == 16 || R == 32, "radix");
    if constexpr (R > 1) {
        C b[R];
#pragma unroll
        for (int i = 0; i < R; ++i) b[i] = a[bitrev<R>(i)];
        dft_levels<DIR, 2, R>(b);
#pragma unroll
        for (int i = 0; i < R; ++i) a[i] = b[i];
    }
}

} // namespace fdas
