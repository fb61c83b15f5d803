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

// One radix-2 DIT butterfly with the compile-time twiddle exp(DIR * 2 pi i * J / LEN):
//   e' = e + w o,  o' = e - w o.     J in [0, LEN/2), LEN in {2,4,8,16,32}
template <int DIR, int J, int LEN>
FDAS_HD void bfly(float2 &e, float2 &o)
{
    constexpr int idx = J * (32 / LEN); // angle = 2 pi idx / 32, idx in [0,16)
    float2 t;
    if constexpr (idx == 0) {
        t = o;
    } else if constexpr (idx == 8) { // w = DIR * i
        t = (DIR > 0) ? make_float2(-o.y, o.x) : make_float2(o.y, -o.x);
    } else if constexpr (idx == 4) { // w = (1 + DIR i)/sqrt2
        constexpr float c = cos32(4);
        t = (DIR > 0) ? make_float2(c * (o.x - o.y), c * (o.x + o.y))
                      : make_float2(c * (o.x + o.y), c * (o.y - o.x));
    } else if constexpr (idx == 12) { // w = (-1 + DIR i)/sqrt2
        constexpr float c = cos32(4);
        t = (DIR > 0) ? make_float2(-c * (o.x + o.y), c * (o.x - o.y))
                      : make_float2(c * (o.y - o.x), -c * (o.x + o.y));
    } else {
        constexpr float wr = cosw(idx);
        constexpr float wi = (DIR > 0) ? sinw(idx) : -sinw(idx);
        t = make_float2(wr * o.x - wi * o.y, wr * o.y + wi * o.x);
    }
    const float2 ee = e;
    e = cadd(ee, t);
    o = csub(ee, t);
}

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

template <int DIR, int LEN, int G, int J, int R>
FDAS_HD void dft_level_j(float2 (&b)[R])
{
    if constexpr (J < LEN / 2) {
        bfly<DIR, J, LEN>(b[G + J], b[G + J + LEN / 2]);
        dft_level_j<DIR, LEN, G, J + 1, R>(b);
    }
}
template <int DIR, int LEN, int G, int R>
FDAS_HD void dft_level_g(float2 (&b)[R])
{
    if constexpr (G < R) {
        dft_level_j<DIR, LEN, G, 0, R>(b);
        dft_level_g<DIR, LEN, G + LEN, R>(b);
    }
}
template <int DIR, int LEN, int R>
FDAS_HD void dft_levels(float2 (&b)[R])
{
    if constexpr (LEN <= R) {
        dft_level_g<DIR, LEN, 0, R>(b);
        dft_levels<DIR, LEN * 2, R>(b);
    }
}

// In-register DFT of length R (power of two, <= 32): a[k] <- sum_n a[n] exp(DIR 2 pi i n k / R).
template <int DIR, int R>
FDAS_HD void dft(float2 (&a)[R])
{
    static_assert(R == 1 || R == 2 || R == 4 || R == 8 || R == 16 || R == 32, "radix");
    if constexpr (R > 1) {
        float2 b[R];
#pragma unroll
        for (int i = 0; i < R; ++i) b[i] = a[bitrev<R>(i)];
        dft_levels<DIR, 2, R>(b);
#pragma unroll
        for (int i = 0; i < R; ++i) a[i] = b[i];
    }
}

} // namespace fdas
