// Fused FDAS kernel for segment length 8192 = 2 x 4096 (BASELINE config 4).
//
// A 16-point-per-thread CTA for 8192 points would need 512 threads x <= 128 registers and two
// 128 KB exchange buffers; neither fits.  Instead the 4096-point machinery of fdas_kernel.cuh
// (256 threads, Geo<4096>) runs twice per template slot:
//
//   forward, once per segment (decimation in time over the INPUT parity):
//       Ee = DFT_4096(x[2n]),  Oo = DFT_4096(x[2n+1]),   W = exp(-2 pi i / 8192)
//       X^[k] = Ee[k] + W^k Oo[k],   X^[k+4096] = Ee[k] - W^k Oo[k],   k < 4096
//     both halves go to the thread's 64 words of tensor memory (slot order of Geo<4096>).
//   inverse, per (slot, parity pi) sub-unit (decimation in frequency over the OUTPUT parity):
//       y[2n'+pi] = IDFT_4096( ( (X^H)[k] + (-1)^pi (X^H)[k+4096] ) conj(W)^(pi k) )[n']
//     the Q3 input stage forms the two products (for H and conj H), their sum or
//     twiddled difference, then Q3/Q2/Q1 run as in the 4096 kernel.  H (both halves, 64
//     registers) is loaded once per slot and serves both parities.
//   store: column 2n'+pi of rows -|z| and +|z| (stride-2 streaming stores; the two parities of
//     a slot follow each other in the same CTA, so L2 merges the sectors).
//
// Interbinning (eq. 4) at this segment length: y[n] and y[n+1] belong to different parity
// sub-units, and neither 64 more registers nor 64 KB more shared memory are there to keep one of them.
// The difference is taken in the FREQUENCY domain instead (shift theorem):
//       (pi/4) (y[n] - y[n+1]) = IDFT_8192( X^H[k] * (pi/4)(1 - exp(+2 pi i k / 8192)) )[n]
// so a slot runs two more sub-units ("half" = 1) whose Q3 input stage scales X^ by that factor (the same
// for H and conj H) and whose powers are the half-bin cells P[r+1/2] = (pi/4)^2 |y[r] - y[r+1]|^2.  An
// interbinned 8192 slot therefore costs two plain ones (the paper's own interbinning cost was x1.1-1.6
// on top of the transform; the shuffle epilogue of the smaller segment lengths is x1.4).
//
// X^ (both halves, 64 words per thread, lane-private and read once per sub-unit) lives in TENSOR MEMORY
// (tcgen05.st once per segment, two tcgen05.ld.x16 per eight slots), which frees the 64 KB of shared memory it
// took in round 1: E1 is double-buffered behind one split-phase `full` barrier per buffer, as in fdas_kernel.cuh.
#pragma once
#include "fdas_kernel3.cuh"

namespace fdas {

struct Geo8k {
    using G = Geo<4096>;
    static constexpr int L = 8192;
    static constexpr int TM_COLS = 128;                // tensor memory: X^lo, X^hi (32 words each) per thread, two warp sets
    static constexpr int smem_bytes() { return 32 + (G::E2_ELEMS + 2 * G::E1_ELEMS) * 16; }   // E2, two E1 buffers
};

#ifdef __CUDACC__

// exp(+2 pi i i / 32), i < 16
__device__ __forceinline__ constexpr float c32re(int i) { return cosw(i); }
__device__ __forceinline__ constexpr float c32im(int i) { return sinw(i); }

// Q3 of one parity: products, sum / twiddled difference, inverse DFT16 over k3, twiddle, store E2.
template <int PARITY, int HALF = 0>
__device__ __forceinline__ void inv_q3_8k(uint32_t tmw, const float4 (&hlo)[8],
                                          const float4 (&hhi)[8], float2 wb, const InvTwiddles<4096> &tw,
                                          const ThreadMap<4096> &tm, const XBuf &e2,
                                          const float2 *__restrict__ wtab2 = nullptr)
{
    using G = Geo<4096>;
    cpk a[16];
#pragma unroll
    for (int c = 0; c < 2; ++c) {
    uint32_t wl[16], wh[16];                           // X^lo / X^hi of slots 8c .. 8c+7 from tensor memory
    tmem_ld2(tmw + 16 * c, wl, tmw + 32 + 16 * c, wh);
#pragma unroll
    for (int ii = 0; ii < 8; ++ii) {
        const int i = 8 * c + ii;
        float2 xl = w2f(wl, ii), xh = w2f(wh, ii);
        if constexpr (HALF) {
            // (pi/4)(1 -+ e) with e = exp(+2 pi i k / 8192), k = k1 + 16 k2 + 256 i (the slot of xl; xh is k + 4096)
            constexpr float S = 0.78539816339744830961566084581988f;
            const float2 w = wtab2[tm.k1 + 16 * tm.k2m + 256 * i];          // exp(-2 pi i k / 8192)
            const float2 fl = make_float2(S - S * w.x, S * w.y), fh = make_float2(S + S * w.x, -S * w.y);
            xl = cmul(xl, fl);
            xh = cmul(xh, fh);
        }
        const float4 l4 = hlo[i >> 1], h4 = hhi[i >> 1];
        const float2 hl = (i & 1) ? make_float2(l4.z, l4.w) : make_float2(l4.x, l4.y);
        const float2 hh = (i & 1) ? make_float2(h4.z, h4.w) : make_float2(h4.x, h4.y);
        constexpr float sg = PARITY ? -1.0f : 1.0f;
        // p = xl hl + sg xh hh,  q = xl conj(hl) + sg xh conj(hh)
        const float ac = fmaf(sg * xh.x, hh.x, xl.x * hl.x);
        const float bd = fmaf(sg * xh.y, hh.y, xl.y * hl.y);
        const float bc = fmaf(sg * xh.y, hh.x, xl.y * hl.x);
        const float ad = fmaf(sg * xh.x, hh.y, xl.x * hl.y);
        cpk v;
        v.re = make_float2(ac - bd, ac + bd);
        v.im = make_float2(bc + ad, bc - ad);
        if constexpr (PARITY) {
            v = cmul(v, wb);                                   // conj(W)^(k1 + 16 k2)
        }
        a[i] = v;
    }
    }
    if constexpr (PARITY) {
        // conj(W)^(256 i) = exp(+2 pi i i / 32): compile-time constants
#pragma unroll
        for (int i = 1; i < 16; ++i) a[i] = cmul(a[i], make_float2(c32re(i), c32im(i)));
    }
    dft<+1, 16>(a);
#pragma unroll
    for (int n3 = 0; n3 < 16; ++n3) {
        const cpk v = (n3 > 0) ? cmul(a[n3], tw.tw3[0][n3]) : a[n3];
        e2.put(tm.e2_q3 + G::C * n3, v);
    }
}

// Plain plane, one parity sub-unit: rows N1 .. N1+3 of both transforms, eight 4-byte streaming stores at immediate
// offsets from the two row bases, each row under its own mask bit (the valid rows differ from lane to lane here: the
// overlap in units of n' is a multiple of 16, not of 32).  Row step = 2 Q cells (the other parity sits in between).
template <int N1>
__device__ __forceinline__ void store_rows_8k(const cpk (&y)[16], float *bp, float *bq, unsigned vm)
{
    constexpr int RB = 2 * Geo<4096>::Q * 4;     // bytes between n1 rows
    float2 pw[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) pw[r] = power2(y[N1 + r]);
    asm volatile("{\n\t.reg .pred p0, p1, p2, p3;\n\t.reg .b32 t;\n\t"
                 "and.b32 t, %10, %15;\n\tsetp.ne.u32 p0, t, 0;\n\t"
                 "and.b32 t, %10, %16;\n\tsetp.ne.u32 p1, t, 0;\n\t"
                 "and.b32 t, %10, %17;\n\tsetp.ne.u32 p2, t, 0;\n\t"
                 "and.b32 t, %10, %18;\n\tsetp.ne.u32 p3, t, 0;\n\t"
                 "@p0 st.global.cs.f32 [%0+%11], %2;\n\t@p0 st.global.cs.f32 [%1+%11], %3;\n\t"
                 "@p1 st.global.cs.f32 [%0+%12], %4;\n\t@p1 st.global.cs.f32 [%1+%12], %5;\n\t"
                 "@p2 st.global.cs.f32 [%0+%13], %6;\n\t@p2 st.global.cs.f32 [%1+%13], %7;\n\t"
                 "@p3 st.global.cs.f32 [%0+%14], %8;\n\t@p3 st.global.cs.f32 [%1+%14], %9;\n\t}"
                 ::"l"(bp), "l"(bq), "f"(pw[0].x), "f"(pw[0].y), "f"(pw[1].x), "f"(pw[1].y), "f"(pw[2].x), "f"(pw[2].y),
                   "f"(pw[3].x), "f"(pw[3].y), "r"(vm), "n"(N1 * RB), "n"((N1 + 1) * RB), "n"((N1 + 2) * RB),
                   "n"((N1 + 3) * RB), "n"(1u << N1), "n"(2u << N1), "n"(4u << N1), "n"(8u << N1)
                 : "memory");
}

// BANKS = 2 (two-bin Fourier interpolation, reading R16; plain sub-units only): prm.npairs counts
// template SLOTS, slot = 2 * pair + bank, as in fdas_kernel.cuh: bank 0 fills the even plane columns, bank 1 (the
// templates at half-integer offsets) the odd ones, and bank 1's q transform is the +|z| row shifted by one bin.
// ESYNC (debug, FDAS_DEBUG_E1_SYNC=1 at fdas_plan_create): a CTA barrier in front of every E1 store, i.e. the
// `empty` hand-shake the two-buffer ordering argument below replaces.  A plane that differs between the two
// builds means that argument no longer holds (tests/test_gpu_parity.py::test_seglen_8192_matches_its_e1_sync_build).
template <int MINB, int MODE = 0, bool INTERBIN = false, int BANKS = 1, bool ESYNC = false>
__global__ void __launch_bounds__(256, MINB) fdas_fused_kernel_8k(const KernelParams prm)
{
    using G = Geo<4096>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t *mbar = reinterpret_cast<uint64_t *>(smem_raw);                 // full[0], full[1] (one per E1 buffer)
    float2 *sm = reinterpret_cast<float2 *>(smem_raw + 32);
    const XBuf e2{sm, sm + G::E2_ELEMS};
    float2 *e1base = sm + 2 * G::E2_ELEMS;
    uint32_t *tslot = reinterpret_cast<uint32_t *>(smem_raw + 16);
    const ThreadMap<4096> tm(threadIdx.x);
    const int tid = tm.tid;

    if (tid == 0) {
        mbar_init(&mbar[0], G::T);
        mbar_init(&mbar[1], G::T);
    }
    // X^ (both halves, 64 words per thread) lives in tensor memory: lane-private, read once per sub-unit
    if (tm.warp == 0) tmem_alloc<Geo8k::TM_COLS>(tslot);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tm_base = *tslot;
    const uint32_t tmw = tm_base + ((uint32_t)(32 * (tm.warp & 3)) << 16) + (uint32_t)(tm.warp >> 2) * 64u;

    InvTwiddles<4096> tw;
    load_inv_twiddles<4096>(prm.wtab, tm, tw);
    // conj(W_8192)^(k1 + 16 k2) for this thread's Q3 slots
    float2 wb;
    {
        const float2 w = prm.wtab2[tm.k1 + 16 * tm.k2m];
        wb = make_float2(w.x, -w.y);
    }

    const long long units = prm.nseg * prm.npairs;
    const long long u0 = units * blockIdx.x / gridDim.x;
    const int n = (int)(units * (blockIdx.x + 1) / gridDim.x - u0);
    if (n <= 0) {
        if (tm.warp == 0) tmem_dealloc<Geo8k::TM_COLS>(tm_base);   // the whole CTA is idle
        return;
    }
    long long seg = u0 / prm.npairs;
    int pair = (int)(u0 - seg * prm.npairs);

    float4 hlo[8], hhi[8];
    constexpr size_t HSTRIDE = (size_t)8 * G::T;      // float4 per half
    int hnext = pair, hloaded = 0;
    auto fetch_h = [&]() {
        if (hloaded < n) {
            const float4 *hp = prm.hperm + (size_t)hnext * 2 * HSTRIDE;
#pragma unroll
            for (int i2 = 0; i2 < 8; ++i2) hlo[i2] = __ldg(hp + i2 * G::T + tid);
#pragma unroll
            for (int i2 = 0; i2 < 8; ++i2) hhi[i2] = __ldg(hp + HSTRIDE + i2 * G::T + tid);
            ++hloaded;
            hnext = (hnext + 1 == prm.npairs) ? 0 : hnext + 1;
        }
    };
    fetch_h();

    // useful outputs in units of n' (n = 2n' + parity; overlap and useful are even)
    const int ov2 = prm.overlap >> 1, us2 = prm.useful >> 1;
    unsigned vmask = 0;
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) {
        const int nn = n1 * G::Q + tid;
        if (nn >= ov2 && nn < ov2 + us2) vmask |= 1u << n1;
    }

    unsigned vmask_m1 = 0;                       // BANKS = 2, bank 1, q row, parity 0: bin 2n' - 1
    if constexpr (BANKS == 2) {
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) {
            const int nn = n1 * G::Q + tid - 1;
            if (nn >= ov2 && nn < ov2 + us2) vmask_m1 |= 1u << n1;
        }
    }

    // sub-units of a slot: s = par + 2 half (half = 1: the interbin difference transform)
    constexpr int SUBS = INTERBIN ? 4 : 2;
    constexpr int CS = INTERBIN ? 2 : 1;              // plane columns per bin
#define FDAS_Q3_SUB(PAR, HALF) inv_q3_8k<PAR, HALF>(tmw, hlo, hhi, wb, tw, tm, e2, prm.wtab2)
    // parked (p, q) powers of sub-units 0..2, see the epilogue.  (The same parking for the plain plane -- parity 0
    // waits, parity 1 stores float2 pairs -- measured 4.35 ms against 3.98 ms for the stride-2 stores: not used.)
    float2 held[INTERBIN && MODE == 0 ? 48 : 1];
    bool have_q3 = false;
    const int nsub = SUBS * n;
    for (int c = 0; c < nsub; ++c) {
        const int sub = c % SUBS;
        const XBuf e1{e1base + (c & 1) * 2 * G::E1_ELEMS, e1base + (c & 1) * 2 * G::E1_ELEMS + G::E1_ELEMS};
        const int par = sub & 1, half = sub >> 1;
        if (!have_q3) {
            // first sub-unit of a segment for this CTA (always parity 0): forward transform
            __syncthreads();
            const long long g0 = seg * prm.useful - prm.overlap;
            float2 xe[16], xo[16];
            fwd_f1<4096, 2, 0>(prm.spectrum, prm.nbins, g0, prm.wtab, tm, e1base);
            __syncthreads();
            fwd_f2<4096>(prm.wtab, tm, e1base, e2.re);
            __syncwarp();
            fwd_f3<4096>(tm, e2.re, xe);
            __syncthreads();
            fwd_f1<4096, 2, 1>(prm.spectrum, prm.nbins, g0, prm.wtab, tm, e1base);
            __syncthreads();
            fwd_f2<4096>(prm.wtab, tm, e1base, e2.re);
            __syncwarp();
            fwd_f3<4096>(tm, e2.re, xo);
            __syncthreads();                                   // E1 / E2 are rewritten below
            {
                uint32_t wl[32], wh[32];
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const float2 t = cmul(xo[i], prm.wtab2[tm.k1 + 16 * tm.k2m + 256 * i]);
                    const float2 lo = cadd(xe[i], t), hi = csub(xe[i], t);
                    wl[2 * i] = __float_as_uint(lo.x);
                    wl[2 * i + 1] = __float_as_uint(lo.y);
                    wh[2 * i] = __float_as_uint(hi.x);
                    wh[2 * i + 1] = __float_as_uint(hi.y);
                }
                tmem_st(tmw, wl);
                tmem_st(tmw + 32, wh);
            }
            inv_q3_8k<0>(tmw, hlo, hhi, wb, tw, tm, e2);
            __syncwarp();
        }
        // Q2: load E2, inverse DFT16 over k2, twiddle; E1 must be free before the stores
        {
            cpk a[16];
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) a[k2] = e2.get(tm.e2_q2 + G::S2 * k2);
            dft<+1, 16>(a);
#pragma unroll
            for (int n2 = 0; n2 < 16; ++n2) a[n2] = cmul(a[n2], tw.tw2[n2]);
            // E1[c & 1]: every warp finished loading sub-unit c-2 from it before it arrived for c-1, and this
            // warp has waited for c-1's arrivals -- no `empty` barrier with two buffers.  This holds only while the
            // y[] loads of a sub-unit stay in front of the next mbar_arrive in program order and the segment-start
            // path keeps its leading __syncthreads; ESYNC re-creates the barrier to check that mechanically.
            if constexpr (ESYNC) __syncthreads();
#pragma unroll
            for (int n2 = 0; n2 < 16; ++n2) e1.put(tm.e1_q2 + n2 * G::R3, a[n2]);
        }
        mbar_arrive(&mbar[c & 1]);
        __syncwarp();

        // Q3 of the next sub-unit of the same segment
        have_q3 = (c + 1 < nsub) && (sub + 1 < SUBS || pair + 1 < prm.npairs);
        if (have_q3) {
            if (sub == 0) {
                FDAS_Q3_SUB(1, 0);
            } else if (INTERBIN && sub == 1) {
                FDAS_Q3_SUB(0, 1);
            } else if (INTERBIN && sub == 2) {
                FDAS_Q3_SUB(1, 1);
            } else {
                FDAS_Q3_SUB(0, 0);                             // first sub-unit of the next slot
            }
            if (sub + 2 == SUBS) fetch_h();                    // next slot's H, one sub-unit ahead
        }
        mbar_wait(&mbar[c & 1], (c >> 1) & 1);

        const int bank = BANKS == 2 ? (pair & 1) : 0;
        const int row_p = BANKS == 2 ? (pair >> 1) : pair;
        const int row_q = prm.ntemplates - 1 - row_p;
        const long long col0 = seg * prm.useful - prm.overlap;
        cpk y[16];
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1) y[k1] = e1.get(k1 * G::S1 + tid);
        dft<+1, 16>(y);
        unsigned vm = vmask;
        if (col0 + prm.overlap + prm.useful > prm.nbins) {
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1)
                if (col0 + 2 * (n1 * G::Q + tid) + par >= prm.nbins) vm &= ~(1u << n1);
        }
        if constexpr (INTERBIN && MODE == 0) {
            // The four cells of bin pair n' (columns 4n' + {0,1,2,3} = sub-units {0,2,1,3}) come from four
            // sub-units of the same thread: the first three are parked in local memory (dynamic index -> never
            // in registers; 384 B per thread, L1/L2-resident) and the fourth stores 16 contiguous bytes per row
            // and lane.  Storing each sub-unit on its own (stride-4 floats, 16 sectors per warp request) cost
            // 12.1 ms on config 4 + interbin against 3.98 ms plain.
            if (sub < 3) {
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1) held[sub * 16 + n1] = power2(y[n1]);
            } else {
                unsigned va = vmask, vb = vmask;         // bins 2n' (cells 0, 1) and 2n'+1 (cells 2, 3)
                if (col0 + prm.overlap + prm.useful > prm.nbins) {
#pragma unroll
                    for (int n1 = 0; n1 < 16; ++n1) {
                        if (col0 + 2 * (n1 * G::Q + tid) >= prm.nbins) va &= ~(1u << n1);
                        if (col0 + 2 * (n1 * G::Q + tid) + 1 >= prm.nbins) vb &= ~(1u << n1);
                    }
                }
                float *bp = prm.plane + (size_t)row_p * prm.ncols + (2 * col0 + 4 * tid);
                float *bq = prm.plane + (size_t)row_q * prm.ncols + (2 * col0 + 4 * tid);
                const bool alp = ((reinterpret_cast<uintptr_t>(bp) & 15) == 0);   // odd nbins: rows alternate
                const bool alq = ((reinterpret_cast<uintptr_t>(bq) & 15) == 0);
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1) {
                    const float2 c0 = held[n1], c2 = held[16 + n1], c1 = held[32 + n1], c3 = power2(y[n1]);
                    const unsigned pa = va & (1u << n1), pb = vb & (1u << n1);
                    st_stream4_if(bp + 4 * n1 * G::Q, c0.x, c1.x, c2.x, c3.x, (alp && pb) ? pa : 0u);
                    st_stream2_if(bp + 4 * n1 * G::Q, c0.x, c1.x, (alp && pb) ? 0u : pa);
                    st_stream2_if(bp + 4 * n1 * G::Q + 2, c2.x, c3.x, alp ? 0u : pb);
                    st_stream4_if(bq + 4 * n1 * G::Q, c0.y, c1.y, c2.y, c3.y, (alq && pb) ? pa : 0u);
                    st_stream2_if(bq + 4 * n1 * G::Q, c0.y, c1.y, (alq && pb) ? 0u : pa);
                    st_stream2_if(bq + 4 * n1 * G::Q + 2, c2.y, c3.y, alq ? 0u : pb);
                }
            }
        } else if constexpr (BANKS == 2) {
            // bin n = 2n' + par -> column 2 n + bank in row p; bank 1's q output n is the half-bin cell of bin n - 1
            float *bp = prm.plane + (size_t)row_p * prm.ncols + (2 * (col0 + 2 * tid + par) + bank);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + (2 * (col0 + 2 * tid + par - bank) + bank);
            unsigned vmq = (bank && par == 0) ? vmask_m1 : vmask;
            if (col0 + prm.overlap + prm.useful >= prm.nbins) {
#pragma unroll 1
                for (int n1 = 0; n1 < 16; ++n1)
                    if (col0 + 2 * (n1 * G::Q + tid) + par - bank >= prm.nbins) vmq &= ~(1u << n1);
            }
            if (row_q == row_p) vmq = 0;                       // z = 0 slot: its q row is the p row again
            emit_unit<4096, false, MODE, 4>(prm, y, bp, bq, vm, vmq);
        } else {
            // bin n = 2n' + par -> plane column CS * (col0 + n) + half
            float *bp = prm.plane + (size_t)row_p * prm.ncols + (CS * (col0 + 2 * tid + par) + half);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + (CS * (col0 + 2 * tid + par) + half);
            const unsigned qon = (MODE != 0 && row_q == row_p) ? 0u : ~0u;   // MODE 1: z = 0 cell reported once
            if constexpr (MODE == 0 && !INTERBIN) {
                store_rows_8k<0>(y, bp, bq, vm);
                store_rows_8k<4>(y, bp, bq, vm);
                store_rows_8k<8>(y, bp, bq, vm);
                store_rows_8k<12>(y, bp, bq, vm);
            } else {
                emit_unit<4096, false, MODE, 2 * CS>(prm, y, bp, bq, vm, vm & qon);
            }
        }
        __syncwarp();
        if (sub == SUBS - 1 && ++pair == prm.npairs) {
            pair = 0;
            ++seg;
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (tm.warp == 0) tmem_dealloc<Geo8k::TM_COLS>(tm_base);
}

#undef FDAS_Q3_SUB

#endif // __CUDACC__

} // namespace fdas
