// Fused FDAS kernel, second generation (L = 2048, 4096): the Q3 -> Q2 transpose of the inverse
// transform goes through warp shuffles instead of shared memory.
//
// Why: measured on B200 the kernel is bound by FP32 issue plus the part of
// the load/store-pipe time the hardware cannot hide under it; a conflict-free LDS.64/STS.64 pair
// moves 8 bytes per lane for 3.4 pipe cycles, one SHFL moves 4 bytes per lane for 1.0 and needs
// no store/load round trip.  E2 (half of all exchanged bytes) never leaves a warp, so it can be
// a rotation of registers between the G = 32/C lanes that share k1:
//
//   round r = 0..G-1: lane g hands its column n3 = (g + r) mod G to lane (g + r) mod G.
//
// For the register index to be the compile-time constant r on BOTH sides, the sender must hold
// its DFT_R3 outputs rotated by its own g and the receiver must accept its DFT16 inputs rotated
// by its own g.  Both rotations are free:
//   sender:   out[(g+r) mod R3] = sum_k3 (in[k3] e^{+2 pi i k3 g/R3}) e^{+2 pi i k3 r/R3}: the extra
//             phase is folded into X^ once per segment (the same for the H and conj(H) products);
//   receiver: slot r holds k2m = (g - r) mod G, and
//             sum_r s[r] e^{+2 pi i ((g-r) mod G) n/G} = e^{+2 pi i g n/G} * DFT^-_G(s)[n]:
//             a forward-direction DFT over the slots, the phase folded into the Q2 -> Q1 twiddles.
//   G = 8 (L = 2048, two DFT8 blocks j per thread, k2 = k2m + 8 j): DFT16 = DFT2 over j, twiddle
//             e^{+2 pi i k2m/16} on the odd branch, DFT8 over k2m; with k2m = (g - r) mod 8 that
//             twiddle is e^{2 pi i g/16} e^{-2 pi i r/16} * (-1)^{[r > g]}: a compile-time constant
//             times a per-lane sign (7 registers), the e^{2 pi i g/16} again folded into the twiddles.
//
// Pipeline: with the exchanged values in registers, Q3 and Q2 of one unit run back to back and
// unit c+1 is produced (-> E1[(c+1)&1]) before Q1 of unit c is consumed: two thirds of a unit lie
// between a warp's arrive and its wait on the `full` barrier.  `empty` barriers protect the two
// E1 buffers; the interbin mailbox of unit u-2 is flushed behind the same `empty` wait.
#pragma once
#include "fdas_kernel.cuh"

namespace fdas {

template <int L>
struct Geo2 : Geo<L> {
    using G = Geo<L>;
    static constexpr int GRP = G::KM;                       // lanes per exchange group (= R3)
    static_assert(G::KM == G::R3 && (G::R3 == 8 || G::R3 == 16), "shuffle exchange: L = 2048 or 4096");
    static constexpr int smem_bytes(bool interbin)
    {
        return 32 /* full[2], empty[2] */ + 2 * G::E1_ELEMS * 16 + (interbin ? G::EDGE_ELEMS * 16 : 0) + 16 /* segment barrier */;
    }
};

#ifdef __CUDACC__

template <int L>
struct InvTwiddles2 {
    float2 tw3r[Geo<L>::NB3][Geo<L>::R3]; // [j][r]: exp(+2 pi i k2_j n3 / (16 R3)), n3 = (g + r) mod R3
    float2 tw2p[16];                      // [n2]: exp(+2 pi i k1 (n2 R3 + g) / L) * exp(+2 pi i g n2 / 16)
    float sg[8];                          // R3 == 8: (r > g ? -1 : 1) * gain of the constant twiddle r
};

// compile-time pieces of c_r = exp(-2 pi i r / 16) = gain * (p + i q), (p, q) = (1, t) or (t, 1)
FDAS_HD constexpr float c16_cos(int r) { return cosw(2 * r); }
FDAS_HD constexpr float c16_sin(int r) { return -sinw(2 * r); }
FDAS_HD constexpr bool c16_cos_major(int r) { return r <= 2 || r >= 6; }
FDAS_HD constexpr float c16_gain(int r) { return c16_cos_major(r) ? c16_cos(r) : c16_sin(r); }
FDAS_HD constexpr float c16_t(int r) { return c16_cos_major(r) ? c16_sin(r) / c16_cos(r) : c16_cos(r) / c16_sin(r); }

template <int L>
__device__ __forceinline__ void load_inv_twiddles2(const float2 *__restrict__ wtab, const ThreadMap<L> &tm,
                                                   InvTwiddles2<L> &tw)
{
    using G = Geo<L>;
    const int g = tm.n3;                                    // = k2m: index inside the exchange group
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
        const int k2 = g + G::KM * j;
#pragma unroll
        for (int r = 0; r < G::R3; ++r) {
            const int n3 = (g + r) & (G::R3 - 1);
            const float2 w = wtab[16 * k2 * n3];
            tw.tw3r[j][r] = make_float2(w.x, -w.y);
        }
    }
#pragma unroll
    for (int n2 = 0; n2 < 16; ++n2) {
        const float2 w = wtab[tm.k1 * (n2 * G::R3 + g)];
        const float2 p = wtab[(g * n2 * (L / 16)) & (L - 1)];
        const float2 wp = cmul(w, p);
        tw.tw2p[n2] = make_float2(wp.x, -wp.y);
    }
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        tw.sg[r] = (G::R3 == 8) ? ((r > g) ? -c16_gain(r) : c16_gain(r)) : 0.f;
        if (G::R3 == 8) asm volatile("" : "+f"(tw.sg[r]));   // keep it in a register: do not re-derive per unit
    }
}

// Fold exp(+2 pi i k3 g / R3) into X^ (once per segment): Q3's outputs then come out rotated by g.
template <int L>
__device__ __forceinline__ void rotate_xhat(const float2 *__restrict__ wtab, const ThreadMap<L> &tm,
                                            float2 (&xh)[Geo<L>::PTS])
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB3; ++j)
#pragma unroll
        for (int k3 = 1; k3 < G::R3; ++k3) {
            const float2 w = wtab[(k3 * tm.n3 * (L / G::R3)) & (L - 1)];
            xh[j * G::R3 + k3] = cmul_conj(xh[j * G::R3 + k3], w);
        }
}

// Tail of Q3 (inverse DFT_R3, twiddle), the shuffle exchange, and Q2's DFT16 + twiddle, starting
// from the products a[j][k3].  Returns the 16 values this thread stores to E1 (index n2).
template <int L>
__device__ __forceinline__ void q3_tail_q2(cpk (&a)[Geo<L>::NB3][Geo<L>::R3], const InvTwiddles2<L> &tw,
                                           const ThreadMap<L> &tm, cpk (&out)[16])
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
        dft<+1, G::R3>(a[j]);
#pragma unroll
        for (int r = 0; r < G::R3; ++r) a[j][r] = cmul(a[j][r], tw.tw3r[j][r]);
    }
    // exchange: slot r of lane g goes to lane (g + r) mod G of the same k1 (lane +- C*r mod 32)
#pragma unroll
    for (int r = 1; r < G::R3; ++r) {
        const int src = tm.lane + 32 - G::C * r;            // SHFL.IDX uses the lane modulo 32
#pragma unroll
        for (int j = 0; j < G::NB3; ++j) {
            cpk v;
            v.re.x = __shfl_sync(0xffffffffu, a[j][r].re.x, src);
            v.re.y = __shfl_sync(0xffffffffu, a[j][r].re.y, src);
            v.im.x = __shfl_sync(0xffffffffu, a[j][r].im.x, src);
            v.im.y = __shfl_sync(0xffffffffu, a[j][r].im.y, src);
            a[j][r] = v;                                     // now: k2 = ((g - r) mod G) + KM*j at n3 = g
        }
    }
    if constexpr (G::R3 == 16) {
        dft<-1, 16>(a[0]);
#pragma unroll
        for (int n2 = 0; n2 < 16; ++n2) out[n2] = cmul(a[0][n2], tw.tw2p[n2]);
    } else {
        cpk u0[8], u1[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            u0[r].re = add2(a[0][r].re, a[1][r].re);
            u0[r].im = add2(a[0][r].im, a[1][r].im);
            u1[r].re = sub2(a[0][r].re, a[1][r].re);
            u1[r].im = sub2(a[0][r].im, a[1][r].im);
        }
#pragma unroll
        for (int r = 1; r < 8; ++r) {                       // u1[r] *= sign_r(g) * exp(-2 pi i r / 16)
            const float t = c16_t(r);
            float2 p, q;
            if (c16_cos_major(r)) {                          // gain * (1 + i t)
                p = fma2(bc2(-t), u1[r].im, u1[r].re);
                q = fma2(bc2(t), u1[r].re, u1[r].im);
            } else {                                         // gain * (t + i)
                p = fma2(bc2(t), u1[r].re, neg2(u1[r].im));
                q = fma2(bc2(t), u1[r].im, u1[r].re);
            }
            u1[r].re = mul2(p, bc2(tw.sg[r]));
            u1[r].im = mul2(q, bc2(tw.sg[r]));
        }
        dft<-1, 8>(u0);
        dft<-1, 8>(u1);
#pragma unroll
        for (int nh = 0; nh < 8; ++nh) {
            out[2 * nh] = cmul(u0[nh], tw.tw2p[2 * nh]);
            out[2 * nh + 1] = cmul(u1[nh], tw.tw2p[2 * nh + 1]);
        }
    }
}

// Q3 products p = X^ H, q = X^ conj(H), then q3_tail_q2.
template <int L>
__device__ __forceinline__ void inv_q3_q2(const float2 (&xh)[Geo<L>::PTS], const float4 (&h4)[Geo<L>::PTS / 2],
                                          const InvTwiddles2<L> &tw, const ThreadMap<L> &tm, cpk (&out)[16])
{
    using G = Geo<L>;
    cpk a[G::NB3][G::R3];
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
#pragma unroll
        for (int k3 = 0; k3 < G::R3; ++k3) {
            const int i = j * G::R3 + k3;
            const float4 hh = h4[i >> 1];
            const float2 h = (i & 1) ? make_float2(hh.z, hh.w) : make_float2(hh.x, hh.y);
            const float2 x = xh[i];
            const float ac = x.x * h.x, bc = x.y * h.x;
            a[j][k3].re = make_float2(fmaf(-x.y, h.y, ac), fmaf(x.y, h.y, ac));
            a[j][k3].im = make_float2(fmaf(x.x, h.y, bc), fmaf(-x.x, h.y, bc));
        }
    }
    q3_tail_q2<L>(a, tw, tm, out);
}

template <int L, bool INTERBIN, int MINB, int MODE = 0, int BANKS = 1>   // BANKS = 2: see fdas_kernel.cuh
__global__ void __launch_bounds__(Geo<L>::T, MINB) fdas_fused_kernel2(const KernelParams prm)
{
    using G = Geo<L>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);                 // full[0], full[1]
    uint64_t *empty = full + 2;                                              // empty[0], empty[1]
    float2 *e1base = reinterpret_cast<float2 *>(smem_raw + 32);              // two (re, im) buffers
    float4 *edges = reinterpret_cast<float4 *>(e1base + 4 * G::E1_ELEMS);    // interbin only
    // bulk segment load: transaction barrier in the last 16 bytes of the allocation
    uint64_t *segbar = reinterpret_cast<uint64_t *>(smem_raw + 32 + 2 * G::E1_ELEMS * 16 + (INTERBIN ? G::EDGE_ELEMS * 16 : 0));
    const ThreadMap<L> tm(threadIdx.x);
    const int tid = tm.tid;

    if (tid == 0) {
        mbar_init(&full[0], G::T);
        mbar_init(&full[1], G::T);
        mbar_init(&empty[0], G::T);
        mbar_init(&empty[1], G::T);
        mbar_init(segbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");   // visible to the async proxy
    }
    __syncthreads();

    InvTwiddles2<L> tw;
    load_inv_twiddles2<L>(prm.wtab, tm, tw);

    const long long units = prm.nseg * prm.npairs;
    const long long u0 = units * blockIdx.x / gridDim.x;
    const int n = (int)(units * (blockIdx.x + 1) / gridDim.x - u0);
    if (n <= 0) return;
    long long seg = u0 / prm.npairs;
    int pair = (int)(u0 - seg * prm.npairs);

    float2 xh[G::PTS];
    float4 h4[G::PTS / 2];
    constexpr size_t HSTRIDE = (size_t)(G::PTS / 2) * G::T;
    int hnext = pair, hloaded = 0;                // H is fetched one unit ahead, in unit order
    auto fetch_h = [&]() {
        if (hloaded < n) {
            load_h<L>(prm.hperm + hnext * HSTRIDE, tid, h4);
            ++hloaded;
            hnext = (hnext + 1 == prm.npairs) ? 0 : hnext + 1;
        }
    };
    fetch_h();

    unsigned vmask = 0;
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) {
        const int nn = n1 * G::Q + tid;
        if (nn >= prm.overlap && nn < prm.overlap + prm.useful) vmask |= 1u << n1;
    }

    unsigned vmask_q1 = 0;                       // BANKS = 2, bank 1, q row: output n is bin n - 1
    if constexpr (BANKS == 2) {
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) {
            const int nn = n1 * G::Q + tid - 1;
            if (nn >= prm.overlap && nn < prm.overlap + prm.useful) vmask_q1 |= 1u << n1;
        }
    }
    Pending<L> pend[2] = {{0, 0, 0, false}, {0, 0, 1, false}};
    auto e1buf = [&](int u) {
        float2 *b = e1base + (u & 1) * 2 * G::E1_ELEMS;
        return XBuf{b, b + G::E1_ELEMS};
    };
    // Q3 + exchange + Q2 of unit u -> E1[u & 1]
    auto produce = [&](int u) {
        cpk o[16];
        inv_q3_q2<L>(xh, h4, tw, tm, o);
        fetch_h();
        if (u >= 2) mbar_wait(&empty[u & 1], ((u >> 1) - 1) & 1);   // every warp has consumed unit u-2
        if (INTERBIN && pend[u & 1].on) flush_edges<L, MODE>(prm, tm, edges, pend[u & 1]);
        const XBuf e1 = e1buf(u);
#pragma unroll
        for (int n2 = 0; n2 < 16; ++n2) e1.put(tm.e1_q2 + n2 * G::R3, o[n2]);
        mbar_arrive(&full[u & 1]);
    };

    // Consume unit q (E1[q & 1] -> Q1 -> power -> plane), `qpair` = its template slot.
    auto consume = [&](int q, int qpair) {
        mbar_wait(&full[q & 1], (q >> 1) & 1);                 // all of E1[q & 1] is written
        const XBuf e1 = e1buf(q);
        const int bank = BANKS == 2 ? (qpair & 1) : 0;
        const int row_p = BANKS == 2 ? (qpair >> 1) : qpair;   // z <= 0
        const int row_q = prm.ntemplates - 1 - row_p;   // z >= 0 (same row for the z = 0 slot)
        const long long col0 = seg * prm.useful - prm.overlap;  // column of local index 0
        const unsigned qon = (MODE != 0 && row_q == row_p) ? 0u : ~0u;   // MODE 1: z = 0 cell reported once
        cpk y[16];
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1) y[k1] = e1.get(k1 * G::S1 + tid);
        if constexpr (!INTERBIN) mbar_arrive(&empty[q & 1]);
        dft<+1, 16>(y);
        // columns >= nbins (last segment): outputs n1 >= ceil((nbins - col0 - tid) / Q) are dropped
        unsigned vm = vmask;
        unsigned vmq = bank ? vmask_q1 : vmask;
        if (col0 + prm.overlap + prm.useful >= prm.nbins) {
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) {
                if (col0 + n1 * G::Q + tid >= prm.nbins) vm &= ~(1u << n1);
                if (col0 + n1 * G::Q + tid - bank >= prm.nbins) vmq &= ~(1u << n1);
            }
        }
        if constexpr (BANKS == 2) {
            float *bp = prm.plane + (size_t)row_p * prm.ncols + (2 * (col0 + tid) + bank);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + (2 * (col0 + tid - bank) + bank);
            emit_unit<L, false, MODE, 2>(prm, y, bp, bq, vm, row_q == row_p ? 0u : vmq);
        } else if constexpr (!INTERBIN) {
            float *bp = prm.plane + (size_t)row_p * prm.ncols + (col0 + tid);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + (col0 + tid);
            emit_unit<L, false, MODE, 1>(prm, y, bp, bq, vm, vmq & qon);
        } else {
            const int par = q & 1;
            float4 *eb = edges + par * (2 * G::W * 16) + (tm.lane == 0 ? G::W * 16 : 0) + tm.warp * 16;
            if (tm.lane == 31 || tm.lane == 0) {
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1)
                    eb[n1] = make_float4(y[n1].re.x, y[n1].re.y, y[n1].im.x, y[n1].im.y);
            }
            mbar_arrive(&empty[par]);                          // E1[par] read, mailbox[par] written
            float *bp = prm.plane + (size_t)row_p * prm.ncols + 2 * (col0 + tid);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + 2 * (col0 + tid);
            if (tm.lane == 31) vm = 0;
            emit_unit<L, true, MODE, 1>(prm, y, bp, bq, vm, vm & qon);
            pend[par].col0 = col0;
            pend[par].pair = row_p;
            pend[par].par = par;
            pend[par].on = true;
        }
    };

    // Per unit u: [forward transform at a segment start] produce(u); then consume u-1 (same
    // segment) and, at the end of the segment or of this CTA's range, u itself.  A whole unit of
    // other work lies between a warp's arrive on full[u & 1] and its wait on it.
    unsigned nbulk = 0;                                        // bulk segment loads so far (phase of `segbar`)
    for (int u = 0; u < n; ++u) {
        const bool first = (u == 0) || (pair == 0);
        if (first) {
            __syncthreads();                                   // every earlier unit is consumed
            if (INTERBIN) {
                if (pend[0].on) flush_edges<L, MODE>(prm, tm, edges, pend[0]);
                if (pend[1].on) flush_edges<L, MODE>(prm, tm, edges, pend[1]);
            }
            float2 *scr = e1base + 2 * G::E1_ELEMS;            // second buffer: segment landing zone, then F2 -> F3 scratch
            const long long seg_start = seg * prm.useful - prm.overlap;
            if (seg_start >= 0 && seg_start + L <= prm.nbins) {    // a2: one bulk copy (TMA engine) of the segment
                if (tid == 0) {
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    mbar_expect_tx(segbar, L * (uint32_t)sizeof(float2));
                    bulk_load(scr, prm.spectrum + seg_start, L * (uint32_t)sizeof(float2), segbar);
                }
                mbar_wait(segbar, nbulk & 1);
                ++nbulk;
                fwd_f1_smem<L>(scr, prm.wtab, tm, e1base);
            } else {                                               // first / last segments: zero extension (R7)
                fwd_f1<L>(prm.spectrum, prm.nbins, seg_start, prm.wtab, tm, e1base);
            }
            __syncthreads();
            fwd_f2<L>(prm.wtab, tm, e1base, scr);
            __syncwarp();
            fwd_f3<L>(tm, scr, xh);
            rotate_xhat<L>(prm.wtab, tm, xh);
            __syncthreads();
        }
        produce(u);
        const bool last = (u == n - 1) || (pair + 1 == prm.npairs);
        for (int q = first ? u : u - 1; q <= (last ? u : u - 1); ++q) consume(q, pair - (u - q));
        if (++pair == prm.npairs) {
            pair = 0;
            ++seg;
        }
    }
    if (INTERBIN) {
        __syncthreads();
        if (pend[0].on) flush_edges<L, MODE>(prm, tm, edges, pend[0]);
        if (pend[1].on) flush_edges<L, MODE>(prm, tm, edges, pend[1]);
    }
}



#endif // __CUDACC__

} // namespace fdas
