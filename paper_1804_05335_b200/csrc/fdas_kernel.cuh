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
// Q3: Y+ = X^ * H, Y- = X^ * conj(H), inverse DFT_R3 over k3, twiddle, store E2.
template <int L>
FDAS_HD void load_h(const float4 *__restrict__ hp, int tid, float4 (&h4)[Geo<L>::PTS / 2])
{
    using G = Geo<L>;
#pragma unroll
    for (int i2 = 0; i2 < G::PTS / 2; ++i2) h4[i2] = hp[i2 * G::T + tid];
}

template <int L>
FDAS_HD void inv_q3(const float2 (&xh)[Geo<L>::PTS], const float4 (&h4)[Geo<L>::PTS / 2],
                    const InvTwiddles<L> &tw, int tid, float4 *s0)
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
        const int b = tid + G::T * j;
        float2 p[G::R3], q[G::R3];
#pragma unroll
        for (int k3 = 0; k3 < G::R3; ++k3) {
            const int i = j * G::R3 + k3;
            const float4 hh = h4[i >> 1];
            const float2 h = (i & 1) ? make_float2(hh.z, hh.w) : make_float2(hh.x, hh.y);
            const float2 x = xh[i];
            const float ac = x.x * h.x, bc = x.y * h.x;
            p[k3] = make_float2(ac - x.y * h.y, bc + x.x * h.y);
            q[k3] = make_float2(ac + x.y * h.y, bc - x.x * h.y);
        }
        dft<+1, G::R3>(p);
        dft<+1, G::R3>(q);
#pragma unroll
        for (int n3 = 0; n3 < G::R3; ++n3) {
            float2 pp = p[n3], qq = q[n3];
            if (n3 > 0) {
                pp = cmul(pp, tw.tw3[j][n3]);
                qq = cmul(qq, tw.tw3[j][n3]);
            }
            s0[b + 256 * n3] = make_float4(pp.x, pp.y, qq.x, qq.y);
        }
    }
}

// Q2: load E2, inverse DFT16 over k2, twiddle, store E1.
template <int L>
FDAS_HD void inv_q2(const InvTwiddles<L> &tw, int tid, const float4 *s0, float4 *s1)
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB2; ++j) {
        const int u = tid + G::T * j, k1 = u & 15, n3 = u >> 4;
        float2 p[16], q[16];
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
            const float4 v = s0[k1 + 16 * k2 + 256 * n3];
            p[k2] = make_float2(v.x, v.y);
            q[k2] = make_float2(v.z, v.w);
        }
        dft<+1, 16>(p);
        dft<+1, 16>(q);
#pragma unroll
        for (int n2 = 0; n2 < 16; ++n2) {
            const float2 pp = cmul(p[n2], tw.tw2[j][n2]);
            const float2 qq = cmul(q[n2], tw.tw2[j][n2]);
            s1[k1 * G::S1 + n2 * G::R3 + n3] = make_float4(pp.x, pp.y, qq.x, qq.y);
        }
    }
}

// Q1: load E1, inverse DFT16 over k1 -> y[n1*Q + t1] for butterfly j.
template <int L>
FDAS_HD void inv_q1(int tid, int j, const float4 *s1, float2 (&p)[16], float2 (&q)[16])
{
    using G = Geo<L>;
    const int t1 = tid + G::T * j;
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        const float4 v = s1[k1 * G::S1 + t1];
        p[k1] = make_float2(v.x, v.y);
        q[k1] = make_float2(v.z, v.w);
    }
    dft<+1, 16>(p);
    dft<+1, 16>(q);
}

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

// Persistent fused kernel.  Work = nseg * npairs (segment, template-slot) units, split into
// gridDim.x equal contiguous ranges (segment-major), so each CTA redoes at most one extra
// forward FFT at a range boundary and every CTA gets the same number of inverse FFT pairs.
template <int L, bool INTERBIN, int MINB>
__global__ void __launch_bounds__(Geo<L>::T, MINB) fdas_fused_kernel(const KernelParams prm)
{
    using G = Geo<L>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *s0 = reinterpret_cast<float4 *>(smem_raw);           // E2, L elements
    float4 *s1 = s0 + G::E2_ELEMS;                               // E1, L+16 elements
    float4 *s2 = s1 + G::E1_ELEMS;                               // interbin only, L elements
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
            fwd_f1<L>(prm.spectrum, prm.nbins, seg * prm.useful - prm.overlap, prm.wtab, tid,
                      reinterpret_cast<float2 *>(s1));
            __syncthreads();
            fwd_f2<L>(prm.wtab, tid, reinterpret_cast<const float2 *>(s1),
                      reinterpret_cast<float2 *>(s0));
            __syncthreads();
            fwd_f3<L>(tid, reinterpret_cast<const float2 *>(s0), xh);
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
        const bool has_q = row_q != row_p;
        const long long col0 = seg * prm.useful - prm.overlap;  // column of local index 0
        const bool interior = col0 + prm.overlap + prm.useful <= prm.nbins;

        float2 p[16], q[16];
        inv_q1<L>(tid, 0, s1, p, q);
        if constexpr (!INTERBIN) {
            float *bp = prm.plane + (size_t)row_p * prm.ncols + (col0 + tid);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + (col0 + tid);
            unsigned vm = vmask;
            if (!interior) {
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1)
                    if (col0 + n1 * G::Q + tid >= prm.nbins) vm &= ~(1u << n1);
            }
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1)
                if (vm & (1u << n1)) st_stream(bp + n1 * G::Q, power(p[n1]));
            if (has_q) {
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1)
                    if (vm & (1u << n1)) st_stream(bq + n1 * G::Q, power(q[n1]));
            }
        } else {
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1)
                s2[n1 * G::Q + tid] = make_float4(p[n1].x, p[n1].y, q[n1].x, q[n1].y);
            __syncthreads();
            float *bp = prm.plane + (size_t)row_p * prm.ncols + 2 * (col0 + tid);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + 2 * (col0 + tid);
            unsigned vm = vmask;
            if (!interior) {
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1)
                    if (col0 + n1 * G::Q + tid >= prm.nbins) vm &= ~(1u << n1);
            }
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) {
                if (vm & (1u << n1)) {
                    const float4 nx = s2[n1 * G::Q + tid + 1]; // n + 1 <= overlap + useful < L
                    const float2 dp = make_float2(p[n1].x - nx.x, p[n1].y - nx.y);
                    st_stream2(bp + 2 * n1 * G::Q, power(p[n1]), IB * power(dp));
                    if (has_q) {
                        const float2 dq = make_float2(q[n1].x - nx.z, q[n1].y - nx.w);
                        st_stream2(bq + 2 * n1 * G::Q, power(q[n1]), IB * power(dq));
                    }
                }
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
