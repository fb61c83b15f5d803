// Fused FDAS kernel, third generation.  L = 2048 (BASELINE configs 2 and 5): X^ and twiddles in tensor memory,
// three CTAs per SM.  L = 4096 interbinned (config 3): the same kernel with those values in registers, one CTA per SM.
//
// What round 1 measured (profiles/r1e_*): two warps per SM sub-partition at 237-255
// registers, FMA pipe 47-59 % busy, the SM's load/store data pipe 69-72 % busy, and the issue slot idle more
// than half of the time behind fixed-latency, shared-memory and L2 waits that two warps cannot cover.  Of
// those registers only 64 hold the transform's data; 96 hold values that are private to the thread and
// read-only for a whole segment (X^) or for the whole launch (the inverse twiddles).
//
// This kernel keeps the second generation's structure (fdas_kernel2.cuh: Q3 -> Q2 transpose by warp
// shuffles, produce / consume pipeline over a double-buffered E1) and changes four things:
//
//   1. X^ and the inverse twiddles live in TENSOR MEMORY (256 KB per SM, lane-private in the 32x32b shape
//      like a register file; tcgen05.st once per segment / launch, tcgen05.ld 16-32 words at a time just
//      before use: 784 B/clk/SM measured, profiles/r1e_tmem_probe.md, against 128 B/clk for shared
//      memory).  The kernel needs <= 168 registers, so THREE CTAs (L = 2048) share an SM: three warps
//      per sub-partition in independent phases instead of two.
//   2. L = 2048: a thread owns the ADJACENT pair k2 = 2g + j (not g + 8j) of Q3's columns.  After the
//      rotation exchange the receiving lane holds k2 = 2((g - r) mod 8) + j in slot (j, r), and
//          Z[n + 8p] = e^{2 pi i g n/8} ( B_0[n] + (-1)^p e^{2 pi i n/16} B_1[n] ),
//          B_j = forward-direction DFT8 of slot row j,
//      so the last radix-2 level has compile-time twiddles again (the g + 8j ownership needed a per-lane
//      sign on the odd branch: +40 packed instructions per unit in fdas_kernel2.cuh).  The phase
//      e^{2 pi i g n/8} is folded into the Q2 -> Q1 twiddles.
//   3. Plane stores take their n1 offset as an immediate of the store instruction (one base address per
//      row instead of a 64-bit add per cell); interbinned rows go out four at a time under one predicate.
//   4. The segment is fetched by ONE bulk copy of the TMA engine (cp.async.bulk + mbarrier transaction count)
//      into the free E1 buffer (the segment goes to shared memory once); the first and last
//      segments of a spectrum, which need the zero extension, keep the predicated loads.
//
// Measured effect of each change: DESIGN.md sections 4.2c and 6.
//
// Index maps (as fdas_kernel.cuh): n = n1 Q + n2 R3 + n3, k = k1 + 16 k2 + 256 k3; a warp owns C values
// of k1, lane = k1l + C g, g < G = R3.  Q3: thread (k1, g) holds k2 = NB3 g + j, all k3.  Q2: thread
// (k1, n3 = g) holds all k2.  Q1: thread t1 = n2 R3 + n3 holds all k1.
#pragma once
#include "fdas_kernel.cuh"

namespace fdas {

template <int L>
struct Geo3 : Geo<L> {
    using G = Geo<L>;
    static_assert(G::KM == G::R3 && (G::R3 == 8 || G::R3 == 16), "shuffle exchange: L = 2048 or 4096");
    static constexpr int WSETS = G::W / 4;                 // warps that share a tensor-memory lane quadrant
    static constexpr int TM_XH = 0, TM_TW3 = 32, TM_TW2 = 64, TM_WORDS = 96;   // 32-bit columns per warp
    static constexpr int TM_COLS = WSETS * TM_WORDS <= 128 ? 128 : 256;        // power of two >= 32
    static constexpr int HDR = 64;                         // full[2], empty[2], tensor-memory base slot
    static constexpr int smem_bytes(bool interbin)
    {
        return HDR + 2 * G::E1_ELEMS * 16 + (interbin ? G::EDGE_ELEMS * 16 : 0);
    }
};

// Index of X^'s frequency f in the per-thread register layout of this kernel: returns (tid, i).
template <int L>
FDAS_HD void freq_to_reg3(int f, int &tid, int &i)
{
    using G = Geo<L>;
    const int k1 = f & 15, k2 = (f >> 4) & 15, k3 = f >> 8;
    const int w = k1 / G::C, k1l = k1 % G::C;
    const int g = k2 / G::NB3, j = k2 % G::NB3;
    tid = 32 * w + k1l + G::C * g;
    i = j * G::R3 + k3;
}

// F3 for this ownership: load the F2 scratch over n3, DFT_R3 -> X^ (i = j R3 + k3, k2 = NB3 g + j).
template <int L>
FDAS_HD void fwd_f3_v3(const ThreadMap<L> &tm, const float2 *e2, float2 (&xh)[Geo<L>::PTS])
{
    using G = Geo<L>;
    const int base = tm.warp * G::E2W + (tm.lane % G::C) + G::S2 * G::NB3 * tm.k2m;
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
        float2 a[G::R3];
#pragma unroll
        for (int n3 = 0; n3 < G::R3; ++n3) a[n3] = e2[base + G::S2 * j + G::C * n3];
        dft<-1, G::R3>(a);
#pragma unroll
        for (int k3 = 0; k3 < G::R3; ++k3) xh[j * G::R3 + k3] = a[k3];
    }
}

#ifdef __CUDACC__

// ------------------------------------------------------------------ tensor memory as a register-file extension
#define FDAS_L8(v, o) "=r"(v[o]), "=r"(v[o + 1]), "=r"(v[o + 2]), "=r"(v[o + 3]), "=r"(v[o + 4]), "=r"(v[o + 5]), "=r"(v[o + 6]), "=r"(v[o + 7])
#define FDAS_S8(v, o) "r"(v[o]), "r"(v[o + 1]), "r"(v[o + 2]), "r"(v[o + 3]), "r"(v[o + 4]), "r"(v[o + 5]), "r"(v[o + 6]), "r"(v[o + 7])

template <int COLS>
__device__ __forceinline__ void tmem_alloc(uint32_t *slot)            // one whole warp
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                 ::"r"(smem_u32(slot)), "n"(COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int COLS>
__device__ __forceinline__ void tmem_dealloc(uint32_t base)           // the same warp
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "n"(COLS) : "memory");
}
// 32x32b: lane i of the warp <-> tensor-memory lane (quadrant base + i), one word per column.
// The load and its wait are ONE asm statement, so no consumer of v[] can be scheduled in between.
__device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n\t"
                 "tcgen05.wait::ld.sync.aligned;"
                 : FDAS_L8(v, 0), FDAS_L8(v, 8) : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                 "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n\t"
                 "tcgen05.wait::ld.sync.aligned;"
                 : FDAS_L8(v, 0), FDAS_L8(v, 8), FDAS_L8(v, 16), FDAS_L8(v, 24) : "r"(taddr));
}
// two 16-word loads, one wait
__device__ __forceinline__ void tmem_ld2(uint32_t ta, uint32_t (&a)[16], uint32_t tb, uint32_t (&b)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%32];\n\t"
                 "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%33];\n\t"
                 "tcgen05.wait::ld.sync.aligned;"
                 : FDAS_L8(a, 0), FDAS_L8(a, 8), FDAS_L8(b, 0), FDAS_L8(b, 8) : "r"(ta), "r"(tb));
}
__device__ __forceinline__ void tmem_st(uint32_t taddr, const uint32_t (&v)[32])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
                 "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};\n\t"
                 "tcgen05.wait::st.sync.aligned;"
                 ::"r"(taddr), FDAS_S8(v, 0), FDAS_S8(v, 8), FDAS_S8(v, 16), FDAS_S8(v, 24) : "memory");
}
__device__ __forceinline__ float2 w2f(const uint32_t *v, int i)
{
    return make_float2(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1]));
}

// The thread's 96 read-mostly words (X^, inverse twiddles): tensor memory when PARK, else plain registers (one CTA
// per SM has the registers to spare and two warps per sub-partition cannot cover the tcgen05.ld latency).
template <bool PARK>
struct Words96 {
    uint32_t r[PARK ? 1 : 96];
    uint32_t tmw;
    template <int N>
    __device__ __forceinline__ void get(int off, uint32_t (&v)[N]) const
    {
        if constexpr (PARK) {
            tmem_ld(tmw + off, v);
        } else {
#pragma unroll
            for (int i = 0; i < N; ++i) v[i] = r[off + i];
        }
    }
    __device__ __forceinline__ void put(int off, const uint32_t (&v)[32])
    {
        if constexpr (PARK) {
            tmem_st(tmw + off, v);
        } else {
#pragma unroll
            for (int i = 0; i < 32; ++i) r[off + i] = v[i];
        }
    }
};

// ------------------------------------------------------------------ plane stores
// Power (a6), interbin (a7) and plane store (a8) of this thread's 16 outputs y[n1 Q + tid] of the (p, q) pair;
// bp / bq: address of the n1 = 0 cell in rows p / q, the n1 step is STRIDE Q cells (2 Q interbinned).
// The stores are plain `if (...) __stcs(...)` so that the compiler keeps loop-invariant predicates in predicate
// registers and folds the n1 offsets into the store's immediate (the inline-asm stores of fdas_kernel.cuh cost a
// 64-bit address add, a mask test and a SETP per cell).
template <int L, bool INTERBIN, int STRIDE>
__device__ __forceinline__ void store_cell3(const cpk (&y)[16], int n1, float *bp, float *bq, bool okp, bool okq)
{
    constexpr int Q = Geo<L>::Q;
    constexpr float IB = 0.61685027506808491367715568749226f; // (pi/4)^2, eq. 4 squared
    const float2 pw = power2(y[n1]);
    if constexpr (!INTERBIN) {
        if (okp) __stcs(bp + STRIDE * n1 * Q, pw.x);
        if (okq) __stcs(bq + STRIDE * n1 * Q, pw.y);
    } else {
        cpk d;                                   // y[n] - y[n+1], neighbour from lane + 1
        d.re = sub2(y[n1].re, make_float2(__shfl_down_sync(0xffffffffu, y[n1].re.x, 1),
                                          __shfl_down_sync(0xffffffffu, y[n1].re.y, 1)));
        d.im = sub2(y[n1].im, make_float2(__shfl_down_sync(0xffffffffu, y[n1].im.x, 1),
                                          __shfl_down_sync(0xffffffffu, y[n1].im.y, 1)));
        const float2 ph = mul2(power2(d), bc2(IB));
        if (okp) __stcs(reinterpret_cast<float2 *>(bp + 2 * n1 * Q), make_float2(pw.x, ph.x));
        if (okq) __stcs(reinterpret_cast<float2 *>(bq + 2 * n1 * Q), make_float2(pw.y, ph.y));
    }
}
// Interbinned cells of one n1 row: (P[n], P[n+1/2]) of the p and the q transform
template <int L>
__device__ __forceinline__ void ib_cells(const cpk &y, float2 &cp, float2 &cq)
{
    constexpr float IB = 0.61685027506808491367715568749226f; // (pi/4)^2, eq. 4 squared
    const float2 pw = power2(y);
    cpk d;                                   // y[n] - y[n+1], neighbour from lane + 1
    d.re = sub2(y.re, make_float2(__shfl_down_sync(0xffffffffu, y.re.x, 1), __shfl_down_sync(0xffffffffu, y.re.y, 1)));
    d.im = sub2(y.im, make_float2(__shfl_down_sync(0xffffffffu, y.im.x, 1), __shfl_down_sync(0xffffffffu, y.im.y, 1)));
    const float2 ph = mul2(power2(d), bc2(IB));
    cp = make_float2(pw.x, ph.x);
    cq = make_float2(pw.y, ph.y);
}
// Four interbinned rows N1..N1+3 of both transforms under ONE per-lane predicate: eight 8-byte streaming stores with
// immediate offsets (a C++ `if` around each store compiles to divergent branches, a predicate per asm store to a
// SETP per cell).  ROWS < 4 stores the first ROWS rows only.
template <int L, int N1, int ROWS>
__device__ __forceinline__ void store_ib_rows(const cpk (&y)[16], float *bp, float *bq, unsigned on)
{
    constexpr int RB = 2 * Geo<L>::Q * 4;    // bytes between n1 rows of an interbinned plane row
    float2 cp[4], cq[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        if (r < ROWS) ib_cells<L>(y[N1 + r], cp[r], cq[r]);
        else cp[r] = cq[r] = make_float2(0.f, 0.f);
    }
    asm volatile("{\n\t.reg .pred pp;\n\tsetp.ne.u32 pp, %18, 0;\n\t"
                 "@pp st.global.cs.v2.f32 [%0+%19], {%2, %3};\n\t"
                 "@pp st.global.cs.v2.f32 [%1+%19], {%4, %5};\n\t"
                 ".reg .pred p1;\n\tsetp.ne.and.u32 p1, %23, 0, pp;\n\t"
                 "@p1 st.global.cs.v2.f32 [%0+%20], {%6, %7};\n\t"
                 "@p1 st.global.cs.v2.f32 [%1+%20], {%8, %9};\n\t"
                 ".reg .pred p2;\n\tsetp.ne.and.u32 p2, %24, 0, pp;\n\t"
                 "@p2 st.global.cs.v2.f32 [%0+%21], {%10, %11};\n\t"
                 "@p2 st.global.cs.v2.f32 [%1+%21], {%12, %13};\n\t"
                 ".reg .pred p3;\n\tsetp.ne.and.u32 p3, %25, 0, pp;\n\t"
                 "@p3 st.global.cs.v2.f32 [%0+%22], {%14, %15};\n\t"
                 "@p3 st.global.cs.v2.f32 [%1+%22], {%16, %17};\n\t}"
                 ::"l"(bp), "l"(bq), "f"(cp[0].x), "f"(cp[0].y), "f"(cq[0].x), "f"(cq[0].y), "f"(cp[1].x), "f"(cp[1].y),
                   "f"(cq[1].x), "f"(cq[1].y), "f"(cp[2].x), "f"(cp[2].y), "f"(cq[2].x), "f"(cq[2].y), "f"(cp[3].x),
                   "f"(cp[3].y), "f"(cq[3].x), "f"(cq[3].y), "r"(on), "n"(N1 * RB), "n"((N1 + 1) * RB), "n"((N1 + 2) * RB),
                   "n"((N1 + 3) * RB), "n"(ROWS > 1), "n"(ROWS > 2), "n"(ROWS > 3)
                 : "memory");
}
// Common case: every lane of the warp has the same valid rows and rows 1..14 are all valid (overlap <= Q, not the
// spectrum's last segment): rows 1..14 need no per-cell predicate, rows 0 and 15 a warp-uniform one.  `lane_on`:
// per-lane switch (interbinning: lane 31's cells are finished one unit later by flush_edges).
template <int L, bool INTERBIN, int STRIDE>
__device__ __forceinline__ void store_cells3_fast(const cpk (&y)[16], float *bp, float *bq, bool lane_on, bool q_on,
                                                  bool row0, bool row15)
{
    if constexpr (INTERBIN) {
        store_ib_rows<L, 0, 1>(y, bp, bq, lane_on && row0);
        store_ib_rows<L, 1, 4>(y, bp, bq, lane_on);
        store_ib_rows<L, 5, 4>(y, bp, bq, lane_on);
        store_ib_rows<L, 9, 4>(y, bp, bq, lane_on);
        store_ib_rows<L, 13, 2>(y, bp, bq, lane_on);
        store_ib_rows<L, 15, 1>(y, bp, bq, lane_on && row15);
    } else {
        const bool lq = lane_on && q_on;
        store_cell3<L, INTERBIN, STRIDE>(y, 0, bp, bq, lane_on && row0, lq && row0);
#pragma unroll
        for (int n1 = 1; n1 < 15; ++n1) store_cell3<L, INTERBIN, STRIDE>(y, n1, bp, bq, lane_on, lq);
        store_cell3<L, INTERBIN, STRIDE>(y, 15, bp, bq, lane_on && row15, lq && row15);
    }
}
// Any masks (last segment, wide overlaps, the shifted q row of BANKS = 2).
template <int L, bool INTERBIN, int STRIDE>
__device__ __forceinline__ void store_cells3_masked(const cpk (&y)[16], float *bp, float *bq, unsigned vm, unsigned vmq)
{
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1)
        store_cell3<L, INTERBIN, STRIDE>(y, n1, bp, bq, (vm >> n1) & 1u, (vmq >> n1) & 1u);
}

// last radix-2 level of Q2 at R3 = 8: (Z[n], Z[n+8]) = B_0[n] +- e^{2 pi i n/16} B_1[n]
template <int N = 0>
__device__ __forceinline__ void q2_radix2(cpk (&b0)[8], cpk (&b1)[8])
{
    if constexpr (N < 8) {
        bfly<+1, N, 16>(b0[N], b1[N]);
        q2_radix2<N + 1>(b0, b1);
    }
}

template <int L, bool INTERBIN, int MINB, int MODE = 0, int BANKS = 1>   // BANKS = 2: see fdas_kernel.cuh
__global__ void __launch_bounds__(Geo<L>::T, MINB) fdas_fused_kernel3(const KernelParams prm)
{
    using G = Geo<L>;
    using G3 = Geo3<L>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);                 // full[0], full[1]
    uint64_t *empty = full + 2;                                              // empty[0], empty[1]
    uint32_t *tslot = reinterpret_cast<uint32_t *>(smem_raw + 32);
    float2 *e1base = reinterpret_cast<float2 *>(smem_raw + G3::HDR);         // two (re, im) buffers
    float4 *edges = reinterpret_cast<float4 *>(e1base + 4 * G::E1_ELEMS);    // interbin only
    const ThreadMap<L> tm(threadIdx.x);
    const int tid = tm.tid;
    const int g = tm.n3;                                                     // index inside the exchange group

    uint64_t *segbar = reinterpret_cast<uint64_t *>(smem_raw + 40);          // bulk segment load: transaction barrier
    if (tid == 0) {
        mbar_init(&full[0], G::T);
        mbar_init(&full[1], G::T);
        mbar_init(&empty[0], G::T);
        mbar_init(&empty[1], G::T);
        mbar_init(segbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");   // visible to the async proxy
    }
    constexpr bool PARK = MINB >= 3;                                         // X^ / twiddles in tensor memory
    if (PARK && tm.warp == 0) tmem_alloc<G3::TM_COLS>(tslot);
    if (PARK) asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (PARK) asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tm_base = PARK ? *tslot : 0u;
    // this warp's words: lanes of quadrant (warp % 4), columns [(warp / 4) * TM_WORDS, +TM_WORDS)
    Words96<PARK> wd;
    wd.tmw = tm_base + ((uint32_t)(32 * (tm.warp & 3)) << 16) + (uint32_t)(tm.warp >> 2) * G3::TM_WORDS;

    const long long units = prm.nseg * prm.npairs;
    const long long u0 = units * blockIdx.x / gridDim.x;
    const int n = (int)(units * (blockIdx.x + 1) / gridDim.x - u0);

    if (n > 0) {
        long long seg = u0 / prm.npairs;
        int pair = (int)(u0 - seg * prm.npairs);

        // inverse twiddles -> tensor memory, once per launch
        {
            uint32_t w3[32], w2[32];
#pragma unroll
            for (int j = 0; j < G::NB3; ++j) {
                const int k2 = G::NB3 * g + j;
#pragma unroll
                for (int r = 0; r < G::R3; ++r) {          // slot r of Q3's output: n3 = (g + r) mod R3
                    const int n3 = (g + r) & (G::R3 - 1);
                    const float2 w = prm.wtab[16 * k2 * n3];
                    w3[2 * (j * G::R3 + r)] = __float_as_uint(w.x);
                    w3[2 * (j * G::R3 + r) + 1] = __float_as_uint(-w.y);
                }
            }
#pragma unroll
            for (int n2 = 0; n2 < 16; ++n2) {              // exp(+2 pi i k1 (n2 R3 + g) / L) exp(+2 pi i g n2 / R3)
                const float2 w = prm.wtab[tm.k1 * (n2 * G::R3 + g)];
                const float2 p = prm.wtab[(g * n2 * (L / G::R3)) & (L - 1)];
                const float2 wp = cmul(w, p);
                w2[2 * n2] = __float_as_uint(wp.x);
                w2[2 * n2 + 1] = __float_as_uint(-wp.y);
            }
            wd.put(G3::TM_TW3, w3);
            wd.put(G3::TM_TW2, w2);
        }

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
        // interbinning: cells of lane 31 wait in the mailbox of E1 buffer `par` for one unit (flush_edges).  All
        // pending units belong to one segment (everything is flushed at a segment start), so one col0 serves both.
        long long pend_col0 = 0;
        int pend_row0 = 0, pend_row1 = 0;
        unsigned pend_on = 0;                        // bit par
        auto flush = [&](int par) {
            if (INTERBIN && (pend_on >> par) & 1u) {
                Pending<L> pd{pend_col0, par ? pend_row1 : pend_row0, par, true};
                flush_edges<L, MODE>(prm, tm, edges, pd);
                pend_on &= ~(1u << par);
            }
        };
        // rows n1 = 0 and 15 of this warp's outputs (rows 1..14 are valid whenever overlap <= Q), warp-uniform
        const bool fast_ok = prm.overlap <= G::Q && (prm.overlap & 31) == 0;
        const bool row0 = 32 * tm.warp >= prm.overlap;
        const bool row15 = 15 * G::Q + 32 * tm.warp + 32 <= prm.overlap + prm.useful;
        auto e1buf = [&](int u) {
            float2 *b = e1base + (u & 1) * 2 * G::E1_ELEMS;
            return XBuf{b, b + G::E1_ELEMS};
        };

        // Q3 + exchange + Q2 of unit u -> E1[u & 1]
        auto produce = [&](int u) {
            cpk a[G::NB3][G::R3];
#pragma unroll
            for (int j = 0; j < G::NB3; ++j) {         // p = X^ H, q = X^ conj(H)
                uint32_t xw[2 * G::R3];
                wd.get(G3::TM_XH + 2 * G::R3 * j, xw);
#pragma unroll
                for (int k3 = 0; k3 < G::R3; ++k3) {
                    const int i = j * G::R3 + k3;
                    const float4 hh = h4[i >> 1];
                    const float2 h = (i & 1) ? make_float2(hh.z, hh.w) : make_float2(hh.x, hh.y);
                    const float2 x = w2f(xw, k3);
                    const float ac = x.x * h.x, bc = x.y * h.x;
                    a[j][k3].re = make_float2(fmaf(-x.y, h.y, ac), fmaf(x.y, h.y, ac));
                    a[j][k3].im = make_float2(fmaf(x.x, h.y, bc), fmaf(-x.x, h.y, bc));
                }
            }
            fetch_h();
#pragma unroll
            for (int j = 0; j < G::NB3; ++j) {
                dft<+1, G::R3>(a[j]);
                uint32_t tw[2 * G::R3];
                wd.get(G3::TM_TW3 + 2 * G::R3 * j, tw);
#pragma unroll
                for (int r = 0; r < G::R3; ++r) a[j][r] = cmul(a[j][r], w2f(tw, r));
            }
            // exchange: slot r of lane g goes to lane (g + r) mod G of the same k1 (lane +- C r mod 32)
#pragma unroll
            for (int r = 1; r < G::R3; ++r) {
                const int src = tm.lane + 32 - G::C * r;        // SHFL.IDX uses the lane modulo 32
#pragma unroll
                for (int j = 0; j < G::NB3; ++j) {
                    cpk v;
                    v.re.x = __shfl_sync(0xffffffffu, a[j][r].re.x, src);
                    v.re.y = __shfl_sync(0xffffffffu, a[j][r].re.y, src);
                    v.im.x = __shfl_sync(0xffffffffu, a[j][r].im.x, src);
                    v.im.y = __shfl_sync(0xffffffffu, a[j][r].im.y, src);
                    a[j][r] = v;                                 // now: k2 = NB3 ((g - r) mod G) + j at n3 = g
                }
            }
            // Q2 over the rotated slots (forward-direction DFT, the phase is in the TM_TW2 twiddles)
            if constexpr (G::R3 == 16) {
                dft<-1, 16>(a[0]);
            } else {
                dft<-1, 8>(a[0]);
                dft<-1, 8>(a[1]);
                q2_radix2(a[0], a[1]);                           // a[p][n] = Z[n + 8 p]
            }
            if (u >= 2) mbar_wait(&empty[u & 1], ((u >> 1) - 1) & 1);   // every warp has consumed unit u-2
            flush(u & 1);
            const XBuf e1 = e1buf(u);
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                uint32_t tw[16];
                wd.get(G3::TM_TW2 + 16 * c, tw);
#pragma unroll
                for (int nn = 0; nn < 8; ++nn) {
                    const int n2 = 8 * c + nn;
                    cpk z;                                       // Z[n2]
                    if constexpr (G::R3 == 16) z = a[0][n2];
                    else z = a[c][nn];
                    e1.put(tm.e1_q2 + n2 * G::R3, cmul(z, w2f(tw, nn)));
                }
            }
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
            // columns >= nbins (the spectrum's last segment): per-cell masks; everywhere else the warp-uniform rows
            const bool tail = col0 + prm.overlap + prm.useful >= prm.nbins;
            if constexpr (INTERBIN) {
                const int par = q & 1;
                float4 *eb = edges + par * (2 * G::W * 16) + (tm.lane == 0 ? G::W * 16 : 0) + tm.warp * 16;
                if (tm.lane == 31 || tm.lane == 0) {
#pragma unroll
                    for (int n1 = 0; n1 < 16; ++n1)
                        eb[n1] = make_float4(y[n1].re.x, y[n1].re.y, y[n1].im.x, y[n1].im.y);
                }
                mbar_arrive(&empty[par]);                          // E1[par] read, mailbox[par] written
                pend_col0 = col0;
                if (par) pend_row1 = row_p; else pend_row0 = row_p;
                pend_on |= 1u << par;
            }
            constexpr int CS = (INTERBIN || BANKS == 2) ? 2 : 1;   // plane columns per bin
            float *bp = prm.plane + (size_t)row_p * prm.ncols + (CS * (col0 + tid) + bank);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + (CS * (col0 + tid - bank) + bank);
            const bool lane_on = !(INTERBIN && tm.lane == 31);
            if (MODE == 0 && BANKS == 1 && fast_ok && !tail) {
                store_cells3_fast<L, INTERBIN, 1>(y, bp, bq, lane_on, true, row0, row15);
            } else {
                unsigned vm = vmask;
                unsigned vmq = bank ? vmask_q1 : vmask;
                if (tail) {
#pragma unroll 1
                    for (int n1 = 0; n1 < 16; ++n1) {
                        if (col0 + n1 * G::Q + tid >= prm.nbins) vm &= ~(1u << n1);
                        if (col0 + n1 * G::Q + tid - bank >= prm.nbins) vmq &= ~(1u << n1);
                    }
                }
                if (!lane_on) vm = vmq = 0;
                if (BANKS == 2 && row_q == row_p) vmq = 0;         // z = 0 slot: its q row is the p row again
                if constexpr (MODE == 0) store_cells3_masked<L, INTERBIN, BANKS == 2 ? 2 : 1>(y, bp, bq, vm, vmq);
                else emit_unit<L, INTERBIN, MODE, BANKS == 2 ? 2 : 1>(prm, y, bp, bq, vm, vmq & qon);
            }
        };

        unsigned nbulk = 0;                                        // bulk segment loads so far (phase of `segbar`)
        // Per unit u: [forward transform at a segment start] produce(u); then consume u-1 (same
        // segment) and, at the end of the segment or of this CTA's range, u itself.
        for (int u = 0; u < n; ++u) {
            const bool first = (u == 0) || (pair == 0);
            if (first) {
                __syncthreads();                                   // every earlier unit is consumed
                flush(0);
                flush(1);
                float2 *scr = e1base + 2 * G::E1_ELEMS;            // second buffer: segment landing zone, then F2 -> F3 scratch
                const long long seg_start = seg * prm.useful - prm.overlap;
                if (seg_start >= 0 && seg_start + L <= prm.nbins) {
                    // a2 (the segment goes to shared memory once): one bulk copy of the L bins by the
                    // TMA engine, completion counted in bytes on `segbar`; every thread waits, then reads its 16 bins
                    if (tid == 0) {
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // earlier generic accesses of `scr`
                        mbar_expect_tx(segbar, L * (uint32_t)sizeof(float2));
                        bulk_load(scr, prm.spectrum + seg_start, L * (uint32_t)sizeof(float2), segbar);
                    }
                    mbar_wait(segbar, nbulk & 1);
                    ++nbulk;
                    fwd_f1_smem<L>(scr, prm.wtab, tm, e1base);
                } else {                                           // first / last segments: zero extension (reading R7)
                    fwd_f1<L>(prm.spectrum, prm.nbins, seg_start, prm.wtab, tm, e1base);
                }
                __syncthreads();
                fwd_f2<L>(prm.wtab, tm, e1base, scr);
                __syncwarp();
                float2 xh[G::PTS];
                fwd_f3_v3<L>(tm, scr, xh);
                // fold exp(+2 pi i k3 g / R3) into X^: Q3's outputs then come out rotated by g
                uint32_t xw[32];
#pragma unroll
                for (int j = 0; j < G::NB3; ++j)
#pragma unroll
                    for (int k3 = 0; k3 < G::R3; ++k3) {
                        const int i = j * G::R3 + k3;
                        float2 x = xh[i];
                        if (k3 > 0) x = cmul_conj(x, prm.wtab[(k3 * g * (L / G::R3)) & (L - 1)]);
                        xw[2 * i] = __float_as_uint(x.x);
                        xw[2 * i + 1] = __float_as_uint(x.y);
                    }
                wd.put(G3::TM_XH, xw);
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
            flush(0);
            flush(1);
        }
    }

    if constexpr (PARK) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tm.warp == 0) tmem_dealloc<G3::TM_COLS>(tm_base);
    }
}

#endif // __CUDACC__

} // namespace fdas
