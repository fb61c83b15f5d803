// Fused FDAS correlation kernel: per overlap-save segment, forward FFT -> for every template
// slot: multiply by H (and conj H) -> inverse FFT -> discard overlap -> power (-> interbin) ->
// plane store.  PAPER.md:105 (steps), :129-131 (fused, +-z conjugate pairs), :170-180 (DIF
// forward / DIT inverse, no re-ordering).  Everything between the segment load and the plane
// store stays in registers and shared memory.
//
// Decomposition (L = 16 * 16 * R3, R3 = L/256; PTS = 16 points per thread, T = L/16 threads):
//   forward (DIF):  n = n1*(L/16) + n2*R3 + n3  ->  k = k1 + 16*k2 + 256*k3
//     F1: DFT16 over n1 (thread <-> t1 = n2*R3+n3), twiddle W_L^{k1*t1}
//     F2: DFT16 over n2 (thread <-> u  = k1 + 16*n3), twiddle W_L^{16*k2*n3}
//     F3: DFT_R3 over n3 (thread <-> b = k1 + 16*k2, 16/R3 butterflies per thread)
//   inverse (DIT) is the exact mirror Q3, Q2, Q1 with conjugate twiddles, so the forward
//   result X^ stays in registers in exactly the layout the inverse starts from, and the
//   inverse ends with thread <-> output bin (coalesced plane stores).
//   Exchange layouts (element units):  E2: k1 + 16*k2 + 256*n3       (size L)
//                                      E1: k1*(L/16 + 1) + t1        (size L + 16, padded)
//   Both are bank-conflict free for the 16-byte (+z, -z) element pairs of the inverse.
#pragma once
#include "fdas_fft.cuh"
#include <stdint.h>

namespace fdas {

template <int L>
struct Geo {
    static constexpr int PTS = 16;           // points per thread per transform
    static constexpr int T = L / PTS;        // threads per CTA
    static constexpr int R3 = L / 256;       // radix of the third pass
    static constexpr int NB3 = PTS / R3;     // R3-butterflies per thread in pass 3
    static constexpr int NB2 = PTS / 16;     // 16-butterflies per thread in pass 2
    static constexpr int NB1 = PTS / 16;     // 16-butterflies per thread in pass 1
    static constexpr int Q = L / 16;         // stride of n1 / number of t1 values
    static constexpr int S1 = Q + 1;         // padded row length of exchange E1
    static constexpr int E2_ELEMS = L;
    static constexpr int E1_ELEMS = 16 * S1;
    static constexpr int IB_ELEMS = L + 2;   // interbin neighbour exchange (index L is read, never used)
    static_assert(L == 1024 || L == 2048 || L == 4096, "segment length");
};

// Index of X^'s frequency f in the per-thread register layout: returns (tid, i).
template <int L>
FDAS_HD void freq_to_reg(int f, int &tid, int &i)
{
    using G = Geo<L>;
    const int b = f & 255, k3 = f >> 8;
    tid = b % G::T;
    i = (b / G::T) * G::R3 + k3;
}

struct KernelParams {
    const float2 *spectrum;   // N complex64
    float *plane;             // K x ncols
    const float4 *hperm;      // [npairs][PTS/2][T] float4 = 2 complex H values (z <= 0 rows)
    const float2 *wtab;       // exp(-2 pi i j / L), j < L
    long long nbins;
    long long ncols;
    long long nseg;
    int ntemplates;           // K
    int npairs;               // (K+1)/2
    int overlap;              // ov
    int useful;               // B
};

// ------------------------------------------------------------------ forward passes (float2)
template <int L>
FDAS_HD void fwd_f1(const float2 *__restrict__ spectrum, long long nbins, long long seg_start,
                    const float2 *__restrict__ wtab, int tid, float2 *s1)
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB1; ++j) {
        const int t1 = tid + G::T * j;
        float2 a[16];
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) {
            const long long g = seg_start + n1 * G::Q + t1;
            a[n1] = (g >= 0 && g < nbins) ? spectrum[g] : make_float2(0.f, 0.f);
        }
        dft<-1, 16>(a);
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1) {
            const float2 v = (k1 == 0) ? a[0] : cmul(a[k1], wtab[(k1 * t1) & (L - 1)]);
            s1[k1 * G::S1 + t1] = v;
        }
    }
}

template <int L>
FDAS_HD void fwd_f2(const float2 *__restrict__ wtab, int tid, const float2 *s1, float2 *s0)
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB2; ++j) {
        const int u = tid + G::T * j, k1 = u & 15, n3 = u >> 4;
        float2 a[16];
#pragma unroll
        for (int n2 = 0; n2 < 16; ++n2) a[n2] = s1[k1 * G::S1 + n2 * G::R3 + n3];
        dft<-1, 16>(a);
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
            const float2 v = (k2 == 0) ? a[0] : cmul(a[k2], wtab[16 * k2 * n3]);
            s0[k1 + 16 * k2 + 256 * n3] = v;
        }
    }
}

template <int L>
FDAS_HD void fwd_f3(int tid, const float2 *s0, float2 (&xh)[Geo<L>::PTS])
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
        const int b = tid + G::T * j;
        float2 a[G::R3];
#pragma unroll
        for (int n3 = 0; n3 < G::R3; ++n3) a[n3] = s0[b + 256 * n3];
        dft<-1, G::R3>(a);
#pragma unroll
        for (int k3 = 0; k3 < G::R3; ++k3) xh[j * G::R3 + k3] = a[k3];
    }
}

// ------------------------------------------------------------------ inverse twiddles (registers)
template <int L>
struct InvTwiddles {
    float2 tw3[Geo<L>::NB3][Geo<L>::R3]; // [j][n3]: exp(+2 pi i k2_j n3 / (16 R3)); n3 = 0 unused
    float2 tw2[Geo<L>::NB2][16];         // [j][n2]: exp(+2 pi i k1 (n2 R3 + n3) / L)
};

template <int L>
FDAS_HD void load_inv_twiddles(const float2 *__restrict__ wtab, int tid, InvTwiddles<L> &tw)
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
        const int k2 = (tid + G::T * j) >> 4;
#pragma unroll
        for (int n3 = 0; n3 < G::R3; ++n3) {
            const float2 w = wtab[16 * k2 * n3];
            tw.tw3[j][n3] = make_float2(w.x, -w.y);
        }
    }
#pragma unroll
    for (int j = 0; j < G::NB2; ++j) {
        const int u = tid + G::T * j, k1 = u & 15, n3 = u >> 4;
#pragma unroll
        for (int n2 = 0; n2 < 16; ++n2) {
            const float2 w = wtab[k1 * (n2 * G::R3 + n3)];
            tw.tw2[j][n2] = make_float2(w.x, -w.y);
        }
    }
}

// ------------------------------------------------------------------ inverse passes (+z / -z pairs)
#ifdef __CUDACC__
template <int L>
__device__ __forceinline__ void load_h(const float4 *__restrict__ hp, int tid, float4 (&h4)[Geo<L>::PTS / 2])
{
    using G = Geo<L>;
#pragma unroll
    for (int i2 = 0; i2 < G::PTS / 2; ++i2) h4[i2] = hp[i2 * G::T + tid];
}

// Exchange buffer for packed pairs: the (Re p, Re q) and (Im p, Im q) register pairs live in two
// separate 8-byte planes, so every access is one 64-bit LDS/STS straight from/to the register
// pair the packed arithmetic uses (a 16-byte interleaved element costs 4 MOVs per store to line
// the two pairs up in one aligned register quad).  Same index maps, same wavefront count.
struct XBuf {
    float2 *re, *im;
    __device__ __forceinline__ void put(int i, const cpk &a) const
    {
        re[i] = a.re;
        im[i] = a.im;
    }
    __device__ __forceinline__ cpk get(int i) const
    {
        cpk a;
        a.re = re[i];
        a.im = im[i];
        return a;
    }
};

// Q3: p = X^ * H, q = X^ * conj(H) as one packed pair, inverse DFT_R3 over k3,
// twiddle, store E2.
//   (Re p, Re q) = x.re*h.re -+ x.im*h.im,   (Im p, Im q) = x.im*h.re +- x.re*h.im
// (scalar FMUL/FFMA writing straight into the register pairs: 6 lane-ops per point).
template <int L>
__device__ __forceinline__ void inv_q3(const float2 (&xh)[Geo<L>::PTS], const float4 (&h4)[Geo<L>::PTS / 2],
                                       const InvTwiddles<L> &tw, int tid, const XBuf &s0)
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
        const int b = tid + G::T * j;
        cpk a[G::R3];
#pragma unroll
        for (int k3 = 0; k3 < G::R3; ++k3) {
            const int i = j * G::R3 + k3;
            const float4 hh = h4[i >> 1];
            const float2 h = (i & 1) ? make_float2(hh.z, hh.w) : make_float2(hh.x, hh.y);
            const float2 x = xh[i];
            const float ac = x.x * h.x, bc = x.y * h.x;
            a[k3].re = make_float2(fmaf(-x.y, h.y, ac), fmaf(x.y, h.y, ac));
            a[k3].im = make_float2(fmaf(x.x, h.y, bc), fmaf(-x.x, h.y, bc));
        }
        dft<+1, G::R3>(a);
#pragma unroll
        for (int n3 = 0; n3 < G::R3; ++n3) {
            const cpk v = (n3 > 0) ? cmul(a[n3], tw.tw3[j][n3]) : a[n3];
            s0.put(b + 256 * n3, v);
        }
    }
}

// Q2: load E2, inverse DFT16 over k2, twiddle, store E1.
template <int L>
__device__ __forceinline__ void inv_q2(const InvTwiddles<L> &tw, int tid, const XBuf &s0, const XBuf &s1)
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB2; ++j) {
        const int u = tid + G::T * j, k1 = u & 15, n3 = u >> 4;
        cpk a[16];
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) a[k2] = s0.get(k1 + 16 * k2 + 256 * n3);
        dft<+1, 16>(a);
#pragma unroll
        for (int n2 = 0; n2 < 16; ++n2)
            s1.put(k1 * G::S1 + n2 * G::R3 + n3, cmul(a[n2], tw.tw2[j][n2]));
    }
}

// Q1: load E1, inverse DFT16 over k1 -> y[n1*Q + t1] for butterfly j.
template <int L>
__device__ __forceinline__ void inv_q1(int tid, int j, const XBuf &s1, cpk (&a)[16])
{
    using G = Geo<L>;
    const int t1 = tid + G::T * j;
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) a[k1] = s1.get(k1 * G::S1 + t1);
    dft<+1, 16>(a);
}

// (|p|^2, |q|^2)
__device__ __forceinline__ float2 power2(const cpk &y) { return fma2(y.im, y.im, mul2(y.re, y.re)); }
#endif // __CUDACC__

FDAS_HD float power(float2 y) { return y.x * y.x + y.y * y.y; }

#ifdef __CUDACC__

__device__ __forceinline__ void st_stream(float *p, float v)
{
    asm volatile("st.global.cs.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
}
__device__ __forceinline__ void st_stream2(float *p, float a, float b)
{
    asm volatile("st.global.cs.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}
// predicated forms (no branch around the store)
__device__ __forceinline__ void st_stream_if(float *p, float v, unsigned pred)
{
    asm volatile("{\n\t.reg .pred pp;\n\tsetp.ne.u32 pp, %2, 0;\n\t@pp st.global.cs.f32 [%0], %1;\n\t}"
                 ::"l"(p), "f"(v), "r"(pred) : "memory");
}
__device__ __forceinline__ void st_stream2_if(float *p, float a, float b, unsigned pred)
{
    asm volatile("{\n\t.reg .pred pp;\n\tsetp.ne.u32 pp, %3, 0;\n\t@pp st.global.cs.v2.f32 [%0], {%1, %2};\n\t}"
                 ::"l"(p), "f"(a), "f"(b), "r"(pred) : "memory");
}

// Persistent fused kernel.  Work = nseg * npairs (segment, template-slot) units, split into
// gridDim.x equal contiguous ranges (segment-major), so each CTA redoes at most one extra
// forward FFT at a range boundary and every CTA gets the same number of inverse FFT pairs.
template <int L, bool INTERBIN, int MINB>
__global__ void __launch_bounds__(Geo<L>::T, MINB) fdas_fused_kernel(const KernelParams prm)
{
    using G = Geo<L>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *sm = reinterpret_cast<float2 *>(smem_raw);
    const XBuf s0{sm, sm + G::E2_ELEMS};                                             // E2
    const XBuf s1{sm + 2 * G::E2_ELEMS, sm + 2 * G::E2_ELEMS + G::E1_ELEMS};         // E1 (padded)
    const XBuf s2{sm + 2 * (G::E2_ELEMS + G::E1_ELEMS),
                  sm + 2 * (G::E2_ELEMS + G::E1_ELEMS) + G::IB_ELEMS};               // interbin only
    const int tid = threadIdx.x;

    InvTwiddles<L> tw;
    load_inv_twiddles<L>(prm.wtab, tid, tw);

    const long long units = prm.nseg * prm.npairs;
    long long u = units * blockIdx.x / gridDim.x;
    const long long u_end = units * (blockIdx.x + 1) / gridDim.x;
    if (u >= u_end) return;
    long long seg = u / prm.npairs;
    int pair = (int)(u - seg * prm.npairs);
    bool need_fwd = true;
    float2 xh[G::PTS];
    float4 h4[G::PTS / 2];
    constexpr size_t HSTRIDE = (size_t)(G::PTS / 2) * G::T;
    load_h<L>(prm.hperm + pair * HSTRIDE, tid, h4);

    // which of this thread's 16 outputs n = n1*Q + tid fall in the useful range [ov, ov+B)
    static_assert(G::NB1 == 1, "epilogue assumes one Q1 butterfly per thread");
    unsigned vmask = 0;
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) {
        const int n = n1 * G::Q + tid;
        if (n >= prm.overlap && n < prm.overlap + prm.useful) vmask |= 1u << n1;
    }

    constexpr float IB = 0.61685027506808491367715568749226f; // (pi/4)^2, eq. 4 squared

    for (; u < u_end; ++u) {
        if (need_fwd) {
            need_fwd = false;
            __syncthreads(); // previous unit's readers of s1 are done
            fwd_f1<L>(prm.spectrum, prm.nbins, seg * prm.useful - prm.overlap, prm.wtab, tid, s1.re);
            __syncthreads();
            fwd_f2<L>(prm.wtab, tid, s1.re, s0.re);
            __syncthreads();
            fwd_f3<L>(tid, s0.re, xh);
            __syncthreads(); // s0 is rewritten by inv_q3 below
        }
        inv_q3<L>(xh, h4, tw, tid, s0);
        __syncthreads();

        // next unit; its H is fetched now so the L2 latency hides behind Q2/Q1
        int npair = pair + 1;
        long long nseg_ = seg;
        if (npair == prm.npairs) {
            npair = 0;
            ++nseg_;
        }
        if (u + 1 < u_end) load_h<L>(prm.hperm + npair * HSTRIDE, tid, h4);

        inv_q2<L>(tw, tid, s0, s1);
        __syncthreads();

        const int row_p = pair;                         // z <= 0
        const int row_q = prm.ntemplates - 1 - pair;    // z >= 0 (same row for the z = 0 slot)
        const long long col0 = seg * prm.useful - prm.overlap;  // column of local index 0
        const bool interior = col0 + prm.overlap + prm.useful <= prm.nbins;

        cpk y[16];
        inv_q1<L>(tid, 0, s1, y);
        unsigned vm = vmask;
        if (!interior) {
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1)
                if (col0 + n1 * G::Q + tid >= prm.nbins) vm &= ~(1u << n1);
        }
        // The z = 0 slot has row_q == row_p and q == p bit for bit (H_0 is real), so its second
        // store rewrites the same value: no special case.
        if constexpr (!INTERBIN) {
            float *bp = prm.plane + (size_t)row_p * prm.ncols + (col0 + tid);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + (col0 + tid);
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) {
                const float2 pw = power2(y[n1]);
                st_stream_if(bp + n1 * G::Q, pw.x, vm & (1u << n1));
                st_stream_if(bq + n1 * G::Q, pw.y, vm & (1u << n1));
            }
        } else {
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) s2.put(n1 * G::Q + tid, y[n1]);
            __syncthreads();
            float *bp = prm.plane + (size_t)row_p * prm.ncols + 2 * (col0 + tid);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + 2 * (col0 + tid);
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) {
                const cpk nx = s2.get(n1 * G::Q + tid + 1); // n + 1 <= overlap + useful < L
                cpk d;
                d.re = sub2(y[n1].re, nx.re);
                d.im = sub2(y[n1].im, nx.im);
                const float2 pw = power2(y[n1]);
                const float2 ph = mul2(power2(d), bc2(IB));
                st_stream2_if(bp + 2 * n1 * G::Q, pw.x, ph.x, vm & (1u << n1));
                st_stream2_if(bq + 2 * n1 * G::Q, pw.y, ph.y, vm & (1u << n1));
            }
        }
        pair = npair;
        if (nseg_ != seg) {
            seg = nseg_;
            need_fwd = true;
        }
    }
}

#endif // __CUDACC__

} // namespace fdas
