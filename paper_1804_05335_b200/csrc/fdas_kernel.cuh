// Fused FDAS correlation kernel: per overlap-save segment, forward FFT -> for every template
// slot: multiply by H (and conj H) -> inverse FFT -> discard overlap -> power (-> interbin) ->
// plane store.  PAPER.md:105 (steps), :129-131 (fused, +-z conjugate pairs), :170-180 (DIF
// forward / DIT inverse, no re-ordering).  Everything between the segment load and the plane
// store stays in registers and shared memory.
//
// Decomposition (L = 16 * 16 * R3, R3 = L/256; PTS = 16 points per thread, T = L/16 threads,
// W = T/32 warps, C = 16/W values of k1 owned by one warp):
//   forward (DIF):  n = n1*(L/16) + n2*R3 + n3  ->  k = k1 + 16*k2 + 256*k3
//     F1: DFT16 over n1 (thread <-> t1 = n2*R3+n3 = tid), twiddle W_L^{k1*t1}
//     F2: DFT16 over n2 (thread <-> (k1, n3)),            twiddle W_L^{16*k2*n3}
//     F3: DFT_R3 over n3 (thread <-> (k1, k2), 16/R3 butterflies per thread)
//   inverse (DIT) is the exact mirror Q3, Q2, Q1 with conjugate twiddles, so the forward
//   result X^ stays in registers in exactly the layout the inverse starts from, and the
//   inverse ends with thread <-> output bin (coalesced plane stores).
//
// Thread maps (w = warp, lane):
//   F3/Q3: k1 = C*w + (lane % C), k2 = lane / C + (32/C)*j, j < 16/R3    (i = j*R3 + k3)
//   F2/Q2: k1 = C*w + (lane % C), n3 = lane / C
//   F1/Q1: t1 = tid
// so the Q3 -> Q2 exchange (E2) never leaves the warp (only __syncwarp between them), and only
// the Q2 -> Q1 exchange (E1) crosses warps.  E1 is double-buffered and guarded by one
// split-phase mbarrier per buffer: a warp arrives after writing its Q2 results, runs Q3 of the
// NEXT unit, and only then waits -- warps drift apart by up to a third of a unit, so one warp's
// shared-memory phase overlaps another's FMA phase instead of all warps marching in lock step.
//   E2 (per warp):  (lane%C) + C*n3 + (32+C)*k2          (512 + 15C elements, conflict-free)
//   E1:             k1*(L/16 + 16/C) + t1                (conflict-free for both sides)
// Elements are 16-byte (+z, -z) pairs split in two 8-byte planes (Re p, Re q) / (Im p, Im q).
#pragma once
#include "fdas_fft.cuh"
#include <stdint.h>

namespace fdas {

template <int L>
struct Geo {
    static constexpr int PTS = 16;           // points per thread per transform
    static constexpr int T = L / PTS;        // threads per CTA
    static constexpr int W = T / 32;         // warps per CTA
    static constexpr int C = 16 / W;         // k1 values per warp
    static constexpr int KM = 32 / C;        // k2 values per Q3 butterfly index j
    static constexpr int R3 = L / 256;       // radix of the third pass
    static constexpr int NB3 = PTS / R3;     // R3-butterflies per thread in pass 3
    static constexpr int Q = L / 16;         // stride of n1 / number of t1 values
    static constexpr int S1 = Q + 16 / C;    // padded row length of exchange E1
    static constexpr int S2 = 32 + C;        // k2 stride of the per-warp exchange E2
    static constexpr int E2W = 512 + 15 * C;  // elements per warp region of E2
    static constexpr int E2_ELEMS = W * E2W;
    static constexpr int E1_ELEMS = 16 * S1;
    static constexpr int EDGE_ELEMS = 2 * 2 * W * 16;  // interbin: [buf][own|edge][warp][n1] float4
    static_assert(L == 1024 || L == 2048 || L == 4096, "segment length");
    static_assert(NB3 * 2 == C && KM * NB3 == 16, "thread map");
    static constexpr int smem_bytes(bool interbin)
    {
        return 16 /* two mbarriers */ + (E2_ELEMS + 2 * E1_ELEMS) * 16 + (interbin ? EDGE_ELEMS * 16 : 0);
    }
};

// Index of X^'s frequency f in the per-thread register layout: returns (tid, i).
template <int L>
FDAS_HD void freq_to_reg(int f, int &tid, int &i)
{
    using G = Geo<L>;
    const int k1 = f & 15, k2 = (f >> 4) & 15, k3 = f >> 8;
    const int w = k1 / G::C, k1l = k1 % G::C;
    const int j = k2 / G::KM, k2m = k2 % G::KM;
    tid = 32 * w + k1l + G::C * k2m;
    i = j * G::R3 + k3;
}

// One cell of the plane above the threshold (MODE 1; same layout as fdas_candidate in include/fdas.h)
struct Candidate {
    long long col;
    int row;
    float power;
};

struct KernelParams {
    const float2 *spectrum;   // N complex64
    float *plane;             // K x ncols (MODE 1: null; cells are addressed relative to it, never stored)
    Candidate *cands;         // MODE 1: candidate list, `capacity` entries
    unsigned long long *count; // MODE 1: number of cells found (may exceed capacity)
    long long capacity;
    float threshold;          // MODE 1: keep cells with P > threshold
    const float4 *hperm;      // [npairs][PTS/2][T] float4 = 2 complex H values (z <= 0 rows)
    const float2 *wtab;       // exp(-2 pi i j / L), j < L   (seglen 8192: L = 4096 here)
    const float2 *wtab2;      // seglen 8192 only: exp(-2 pi i j / 8192), j < 8192
    long long nbins;
    long long ncols;
    long long nseg;
    int ntemplates;           // K
    int npairs;               // (K+1)/2
    int overlap;              // ov
    int useful;               // B
};

// Per-thread constants of the thread maps above.
template <int L>
struct ThreadMap {
    int tid, warp, lane;
    int k1;        // F2/Q2 and F3/Q3
    int n3;        // F2/Q2
    int k2m;       // F3/Q3: k2 = k2m + KM*j
    int e2_q3;     // E2 element index of (j = 0, n3 = 0) for this thread's Q3 butterflies
    int e2_q2;     // E2 element index of k2 = 0 for this thread's Q2 butterfly
    int e1_q2;     // E1 element index of n2 = 0 for this thread's Q2 butterfly
    FDAS_HD explicit ThreadMap(int t)
    {
        using G = Geo<L>;
        tid = t;
        warp = t >> 5;
        lane = t & 31;
        const int k1l = lane % G::C;
        k1 = G::C * warp + k1l;
        n3 = lane / G::C;
        k2m = lane / G::C;
        e2_q3 = warp * G::E2W + k1l + G::S2 * k2m;
        e2_q2 = warp * G::E2W + lane;
        e1_q2 = k1 * G::S1 + n3;
    }
};

// ------------------------------------------------------------------ forward passes (float2)
// F1: load the segment (zero outside [0, nbins), reading R7), DFT16 over n1, twiddle, store E1.
// STRIDE/OFF: the transform's input n is bin seg_start + STRIDE*n + OFF (8192 = 2 x 4096 path).
template <int L, int STRIDE = 1, int OFF = 0>
FDAS_HD void fwd_f1(const float2 *__restrict__ spectrum, long long nbins, long long seg_start,
                    const float2 *__restrict__ wtab, const ThreadMap<L> &tm, float2 *e1)
{
    using G = Geo<L>;
    const int t1 = tm.tid;
    float2 a[16];
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) {
        const long long g = seg_start + STRIDE * (n1 * G::Q + t1) + OFF;
        a[n1] = (g >= 0 && g < nbins) ? spectrum[g] : make_float2(0.f, 0.f);
    }
    dft<-1, 16>(a);
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        const float2 v = (k1 == 0) ? a[0] : cmul(a[k1], wtab[(k1 * t1) & (L - 1)]);
        e1[k1 * G::S1 + t1] = v;
    }
}

// F2: load E1 over n2, DFT16, twiddle, store E2 (this warp's region only).
template <int L>
FDAS_HD void fwd_f2(const float2 *__restrict__ wtab, const ThreadMap<L> &tm, const float2 *e1, float2 *e2)
{
    using G = Geo<L>;
    float2 a[16];
#pragma unroll
    for (int n2 = 0; n2 < 16; ++n2) a[n2] = e1[tm.e1_q2 + n2 * G::R3];
    dft<-1, 16>(a);
#pragma unroll
    for (int k2 = 0; k2 < 16; ++k2) {
        const float2 v = (k2 == 0) ? a[0] : cmul(a[k2], wtab[16 * k2 * tm.n3]);
        e2[tm.e2_q2 + G::S2 * k2] = v;
    }
}

// F3: load E2 over n3, DFT_R3 -> X^ in registers (i = j*R3 + k3).
template <int L>
FDAS_HD void fwd_f3(const ThreadMap<L> &tm, const float2 *e2, float2 (&xh)[Geo<L>::PTS])
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
        float2 a[G::R3];
#pragma unroll
        for (int n3 = 0; n3 < G::R3; ++n3) a[n3] = e2[tm.e2_q3 + G::S2 * G::KM * j + G::C * n3];
        dft<-1, G::R3>(a);
#pragma unroll
        for (int k3 = 0; k3 < G::R3; ++k3) xh[j * G::R3 + k3] = a[k3];
    }
}

// ------------------------------------------------------------------ inverse twiddles (registers)
template <int L>
struct InvTwiddles {
    float2 tw3[Geo<L>::NB3][Geo<L>::R3]; // [j][n3]: exp(+2 pi i k2_j n3 / (16 R3)); n3 = 0 unused
    float2 tw2[16];                      // [n2]: exp(+2 pi i k1 (n2 R3 + n3) / L)
};

template <int L>
FDAS_HD void load_inv_twiddles(const float2 *__restrict__ wtab, const ThreadMap<L> &tm, InvTwiddles<L> &tw)
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
        const int k2 = tm.k2m + G::KM * j;
#pragma unroll
        for (int n3 = 0; n3 < G::R3; ++n3) {
            const float2 w = wtab[16 * k2 * n3];
            tw.tw3[j][n3] = make_float2(w.x, -w.y);
        }
    }
#pragma unroll
    for (int n2 = 0; n2 < 16; ++n2) {
        const float2 w = wtab[tm.k1 * (n2 * G::R3 + tm.n3)];
        tw.tw2[n2] = make_float2(w.x, -w.y);
    }
}

// ------------------------------------------------------------------ inverse passes (+z / -z pairs)
#ifdef __CUDACC__
template <int L>
__device__ __forceinline__ void load_h(const float4 *__restrict__ hp, int tid, float4 (&h4)[Geo<L>::PTS / 2])
{
    using G = Geo<L>;
#pragma unroll
    for (int i2 = 0; i2 < G::PTS / 2; ++i2) h4[i2] = __ldg(hp + i2 * G::T + tid);
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
// twiddle, store E2 (this warp's region).
//   (Re p, Re q) = x.re*h.re -+ x.im*h.im,   (Im p, Im q) = x.im*h.re +- x.re*h.im
// (scalar FMUL/FFMA writing straight into the register pairs: 6 lane-ops per point).
template <int L>
__device__ __forceinline__ void inv_q3(const float2 (&xh)[Geo<L>::PTS], const float4 (&h4)[Geo<L>::PTS / 2],
                                       const InvTwiddles<L> &tw, const ThreadMap<L> &tm, const XBuf &e2)
{
    using G = Geo<L>;
#pragma unroll
    for (int j = 0; j < G::NB3; ++j) {
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
            e2.put(tm.e2_q3 + G::S2 * G::KM * j + G::C * n3, v);
        }
    }
}

// Q2: load E2 (own warp's region), inverse DFT16 over k2, twiddle, store E1.
template <int L>
__device__ __forceinline__ void inv_q2(const InvTwiddles<L> &tw, const ThreadMap<L> &tm, const XBuf &e2,
                                       const XBuf &e1)
{
    using G = Geo<L>;
    cpk a[16];
#pragma unroll
    for (int k2 = 0; k2 < 16; ++k2) a[k2] = e2.get(tm.e2_q2 + G::S2 * k2);
    dft<+1, 16>(a);
#pragma unroll
    for (int n2 = 0; n2 < 16; ++n2) e1.put(tm.e1_q2 + n2 * G::R3, cmul(a[n2], tw.tw2[n2]));
}

// Q1: load E1, inverse DFT16 over k1 -> y[n1*Q + t1].
template <int L>
__device__ __forceinline__ void inv_q1(const ThreadMap<L> &tm, const XBuf &e1, cpk (&a)[16])
{
    using G = Geo<L>;
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) a[k1] = e1.get(k1 * G::S1 + tm.tid);
    dft<+1, 16>(a);
}

// (|p|^2, |q|^2)
__device__ __forceinline__ float2 power2(const cpk &y) { return fma2(y.im, y.im, mul2(y.re, y.re)); }

__device__ __forceinline__ void st_stream(float *p, float v)
{
    asm volatile("st.global.cs.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
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

// Plane sink.  MODE 0 (fdas_execute): streaming store of the cell.  MODE 1 (fdas_execute_threshold,
// PAPER.md:73 "comparing the resulting Fourier power to a pre-calculated threshold", :331): the plane
// never reaches memory; a cell above the threshold is appended to the candidate list (rare path:
// its row / column are recovered from the address the store would have used).
// What the out-of-line candidate code needs, passed BY VALUE: taking the address of the kernel's parameter struct
// for a call would make the compiler keep a copy of it in local memory and read every prm.x of the main loop from
// there (measured in the interbinned threshold kernels: LDL + long-scoreboard waits on npairs, threshold, ...).
struct CandSink {
    const float *plane;
    Candidate *cands;
    unsigned long long *count;
    long long capacity, ncols;
    float threshold;
};
__device__ __forceinline__ CandSink sink_of(const KernelParams &prm)
{
    return CandSink{prm.plane, prm.cands, prm.count, prm.capacity, prm.ncols, prm.threshold};
}
__device__ __noinline__ void push_candidate(const CandSink s, const float *p, float v)
{
    const long long idx = p - s.plane;
    const long long row = idx / s.ncols;
    const unsigned long long slot = atomicAdd(s.count, 1ull);
    if (slot < (unsigned long long)s.capacity) {
        Candidate c;
        c.col = idx - row * s.ncols;
        c.row = (int)row;
        c.power = v;
        s.cands[slot] = c;
    }
}
template <int MODE>
__device__ __forceinline__ void emit_if(const KernelParams &prm, float *p, float v, unsigned pred)
{
    if constexpr (MODE == 0) {
        st_stream_if(p, v, pred);
    } else {
        if (pred && v > prm.threshold) push_candidate(sink_of(prm), p, v);
    }
}
template <int MODE>
__device__ __forceinline__ void emit2_if(const KernelParams &prm, float *p, float a, float b, unsigned pred)
{
    if constexpr (MODE == 0) {
        st_stream2_if(p, a, b, pred);
    } else {
        if (pred && a > prm.threshold) push_candidate(sink_of(prm), p, a);
        if (pred && b > prm.threshold) push_candidate(sink_of(prm), p + 1, b);
    }
}

// Epilogue of one unit: power (a6) and interbin (a7) of this thread's 16 outputs y[n1*Q + tid] of the
// (p, q) pair, handed to the plane sink (a8).  bp / bq: address of the n1 = 0 cell in rows p / q; the n1
// step is STRIDE*Q cells (2*Q interbinned).  vm / vmq: valid-output masks of the two rows.
// MODE 1 first takes the maximum over the unit's cells and leaves unless some cell of the WARP passes the
// threshold (warp-uniform, so the interbin shuffles of the slow path stay converged): the common case
// costs no branch per cell.  Masked-out cells take part in the maximum; that can only cost time.
template <int L, bool INTERBIN, int MODE, int STRIDE>
__device__ __forceinline__ void emit_cells(const KernelParams &prm, const cpk (&y)[16], float *bp, float *bq,
                                           unsigned vm, unsigned vmq)
{
    constexpr int Q = Geo<L>::Q;
    constexpr float IB = 0.61685027506808491367715568749226f; // (pi/4)^2, eq. 4 squared
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) {
        const float2 pw = power2(y[n1]);
        if constexpr (!INTERBIN) {
            emit_if<MODE>(prm, bp + STRIDE * n1 * Q, pw.x, vm & (1u << n1));
            emit_if<MODE>(prm, bq + STRIDE * n1 * Q, pw.y, vmq & (1u << n1));
        } else {
            cpk d;                                   // y[n] - y[n+1], neighbour from lane + 1
            d.re = sub2(y[n1].re, make_float2(__shfl_down_sync(0xffffffffu, y[n1].re.x, 1),
                                              __shfl_down_sync(0xffffffffu, y[n1].re.y, 1)));
            d.im = sub2(y[n1].im, make_float2(__shfl_down_sync(0xffffffffu, y[n1].im.x, 1),
                                              __shfl_down_sync(0xffffffffu, y[n1].im.y, 1)));
            const float2 ph = mul2(power2(d), bc2(IB));
            emit2_if<MODE>(prm, bp + 2 * n1 * Q, pw.x, ph.x, vm & (1u << n1));
            emit2_if<MODE>(prm, bq + 2 * n1 * Q, pw.y, ph.y, vmq & (1u << n1));
        }
    }
}
// MODE 1 slow path, out of line (its register needs and calls stay out of the main loop); entered by whole
// warps only, so the interbin shuffles are converged.
template <int L, bool INTERBIN, int STRIDE>
__device__ __noinline__ void emit_cells_rare(const CandSink s, const cpk (&y)[16], float *bp, float *bq,
                                             unsigned vm, unsigned vmq)
{
    KernelParams prm;                                   // the fields the candidate sink reads; local to the rare path
    prm.plane = const_cast<float *>(s.plane);
    prm.cands = s.cands;
    prm.count = s.count;
    prm.capacity = s.capacity;
    prm.ncols = s.ncols;
    prm.threshold = s.threshold;
    emit_cells<L, INTERBIN, 1, STRIDE>(prm, y, bp, bq, vm, vmq);
}

template <int L, bool INTERBIN, int MODE, int STRIDE>
__device__ __forceinline__ void emit_unit(const KernelParams &prm, const cpk (&y)[16], float *bp, float *bq,
                                          unsigned vm, unsigned vmq)
{
    if constexpr (MODE == 0) {
        emit_cells<L, INTERBIN, 0, STRIDE>(prm, y, bp, bq, vm, vmq);
    } else {
        constexpr float IB = 0.61685027506808491367715568749226f;
        float2 mx = power2(y[0]);
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) {
            const float2 pw = power2(y[n1]);
            mx = make_float2(fmaxf(mx.x, pw.x), fmaxf(mx.y, pw.y));
            if constexpr (INTERBIN) {
                cpk d;
                d.re = sub2(y[n1].re, make_float2(__shfl_down_sync(0xffffffffu, y[n1].re.x, 1),
                                                  __shfl_down_sync(0xffffffffu, y[n1].re.y, 1)));
                d.im = sub2(y[n1].im, make_float2(__shfl_down_sync(0xffffffffu, y[n1].im.x, 1),
                                                  __shfl_down_sync(0xffffffffu, y[n1].im.y, 1)));
                const float2 ph = mul2(power2(d), bc2(IB));
                mx = make_float2(fmaxf(mx.x, ph.x), fmaxf(mx.y, ph.y));
            }
        }
        if (__any_sync(0xffffffffu, fmaxf(mx.x, mx.y) > prm.threshold)) {
            cpk ys[16];                              // a copy in local memory: y itself stays in registers
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) ys[n1] = y[n1];
            emit_cells_rare<L, INTERBIN, STRIDE>(sink_of(prm), ys, bp, bq, vm, vmq);
        }
    }
}

__device__ __forceinline__ void st_stream4_if(float *p, float a, float b, float c, float d, unsigned pred)
{
    asm volatile("{\n\t.reg .pred pp;\n\tsetp.ne.u32 pp, %5, 0;\n\t@pp st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};\n\t}"
                 ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d), "r"(pred) : "memory");
}

// ---- split-phase CTA barrier on shared memory (mbarrier): arrive now, wait later
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                 "@!p bra WAIT_%=;\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// ------------------------------------------------------------------ bulk copy of a segment (TMA engine, 1-D)
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}"
                 ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// global -> this CTA's shared memory, completion counted in bytes on `bar` (cp.async.bulk: SASS UBLKCP)
__device__ __forceinline__ void bulk_load(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// F1 from a segment already in shared memory: DFT16 over n1, twiddle, store E1 (as fwd_f1 of fdas_kernel.cuh)
// (STRIDE / OFF as fwd_f1: the transform's input n is element STRIDE n + OFF of the segment)
template <int L, int STRIDE = 1, int OFF = 0>
__device__ __forceinline__ void fwd_f1_smem(const float2 *seg, const float2 *__restrict__ wtab, const ThreadMap<L> &tm,
                                            float2 *e1)
{
    using G = Geo<L>;
    const int t1 = tm.tid;
    float2 a[16];
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) a[n1] = seg[STRIDE * (n1 * G::Q + t1) + OFF];
    dft<-1, 16>(a);
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        const float2 v = (k1 == 0) ? a[0] : cmul(a[k1], wtab[(k1 * t1) & (L - 1)]);
        e1[k1 * G::S1 + t1] = v;
    }
}

// Interbin cells whose neighbour y[n+1] lives in another warp (lane 31 of every warp) are finished
// one unit late from the two small "own" / "edge" mailboxes written during Q1.
template <int L>
struct Pending {
    long long col0;
    int pair, par;
    bool on;
};

template <int L, int MODE = 0>
__device__ __forceinline__ void flush_edges(const KernelParams &prm, const ThreadMap<L> &tm, const float4 *edges,
                                            Pending<L> &pd)
{
    using G = Geo<L>;
    constexpr float IB = 0.61685027506808491367715568749226f; // (pi/4)^2, eq. 4 squared
    const int n1 = tm.lane & 15;
    const float4 *eb = edges + pd.par * (2 * G::W * 16);
    const float4 a = eb[tm.warp * 16 + n1];                                   // y[n] of lane 31
    const float4 b = (tm.warp < G::W - 1) ? eb[(G::W + tm.warp + 1) * 16 + n1]  // y[n+1]: next warp's lane 0
                                          : eb[G::W * 16 + min(n1 + 1, 15)];    // ... or thread 0's next n1
    const bool lo = tm.lane < 16;                                             // lanes 0-15: p row, 16-31: q row
    const float ar = lo ? a.x : a.y, ai = lo ? a.z : a.w;
    const float dr = ar - (lo ? b.x : b.y);
    const float di = ai - (lo ? b.z : b.w);
    const float pw = fmaf(ai, ai, ar * ar);
    const float ph = IB * fmaf(di, di, dr * dr);
    const int n = n1 * G::Q + 32 * tm.warp + 31;
    const long long col = pd.col0 + n;
    const int row = lo ? pd.pair : prm.ntemplates - 1 - pd.pair;
    // MODE 1: the z = 0 slot's q row is its p row again -- report it once
    const bool dup = MODE != 0 && !lo && row == pd.pair;
    emit2_if<MODE>(prm, prm.plane + (size_t)row * prm.ncols + 2 * col, pw, ph,
                   n >= prm.overlap && n < prm.overlap + prm.useful && col < prm.nbins && !dup);
    pd.on = false;
}

// Persistent fused kernel.  Work = nseg * npairs (segment, template-slot) units, split into
// gridDim.x equal contiguous ranges (segment-major), so each CTA redoes at most one extra
// forward FFT at a range boundary and every CTA gets the same number of inverse FFT pairs.
// BANKS = 2 (two-bin Fourier interpolation, reading R16): prm.npairs counts template SLOTS,
// slot = 2 * pair + bank; bank 0 holds the usual templates and fills the even plane columns, bank 1 the
// templates sampled at half-integer offsets t[d] = h_z(d - 1/2) and fills the odd columns.  The +-z pairing
// survives with a one-bin shift: conj(H_bank1 of -|z|) = exp(-2 pi i f / L) H_bank1 of +|z| (h is odd about
// 1/2 there), so the q transform's output n is the half-bin cell of bin n - 1.
template <int L, bool INTERBIN, int MINB, int MODE = 0, int BANKS = 1>
__global__ void __launch_bounds__(Geo<L>::T, MINB) fdas_fused_kernel(const KernelParams prm)
{
    using G = Geo<L>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t *mbar = reinterpret_cast<uint64_t *>(smem_raw);                 // full[0], full[1]
    float2 *sm = reinterpret_cast<float2 *>(smem_raw + 16);
    const XBuf e2{sm, sm + G::E2_ELEMS};                                     // per-warp regions
    float2 *e1base = sm + 2 * G::E2_ELEMS;                                   // two (re, im) buffers
    float4 *edges = reinterpret_cast<float4 *>(e1base + 4 * G::E1_ELEMS);    // interbin only
    const ThreadMap<L> tm(threadIdx.x);
    const int tid = tm.tid;

    if (tid == 0) {
        mbar_init(&mbar[0], G::T);
        mbar_init(&mbar[1], G::T);
    }
    __syncthreads();

    InvTwiddles<L> tw;
    load_inv_twiddles<L>(prm.wtab, tm, tw);

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

    // which of this thread's 16 outputs n = n1*Q + tid fall in the useful range [ov, ov+B)
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
    Pending<L> pend{0, 0, 0, false};
    bool have_q3 = false;

    for (int c = 0; c < n; ++c) {
        if (!have_q3) {
            // first unit of a segment for this CTA: the pipeline is drained; forward transform
            __syncthreads();                                  // nobody reads E1 / E2 / edges any more
            if (INTERBIN && pend.on) flush_edges<L, MODE>(prm, tm, edges, pend);
            fwd_f1<L>(prm.spectrum, prm.nbins, seg * prm.useful - prm.overlap, prm.wtab, tm, e1base);
            __syncthreads();
            fwd_f2<L>(prm.wtab, tm, e1base, e2.re);
            __syncwarp();
            fwd_f3<L>(tm, e2.re, xh);
            __syncthreads();                                  // E1[0] is rewritten by Q2 below
            inv_q3<L>(xh, h4, tw, tm, e2);
            fetch_h();
            __syncwarp();
        }
        const int par = c & 1;
        const XBuf e1{e1base + par * 2 * G::E1_ELEMS, e1base + par * 2 * G::E1_ELEMS + G::E1_ELEMS};
        inv_q2<L>(tw, tm, e2, e1);
        mbar_arrive(&mbar[par]);                              // this warp's share of E1[par] is written
        __syncwarp();                                         // ... and its reads of E2 are done

        // Q3 of the next unit (same segment) fills the time until the other warps arrive
        have_q3 = (c + 1 < n) && (pair + 1 < prm.npairs);
        if (have_q3) {
            inv_q3<L>(xh, h4, tw, tm, e2);
            fetch_h();
        }
        mbar_wait(&mbar[par], (c >> 1) & 1);                  // all of E1[par] is written

        if (INTERBIN && pend.on) flush_edges<L, MODE>(prm, tm, edges, pend);   // every warp is past Q1(c-1)

        const int bank = BANKS == 2 ? (pair & 1) : 0;
        const int row_p = BANKS == 2 ? (pair >> 1) : pair;   // z <= 0
        const int row_q = prm.ntemplates - 1 - row_p;   // z >= 0 (same row for the z = 0 slot)
        const long long col0 = seg * prm.useful - prm.overlap;  // column of local index 0
        cpk y[16];
        inv_q1<L>(tm, e1, y);
        unsigned vm = vmask;
        unsigned vmq = bank ? vmask_q1 : vmask;
        if (col0 + prm.overlap + prm.useful >= prm.nbins) {
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) {
                if (col0 + n1 * G::Q + tid >= prm.nbins) vm &= ~(1u << n1);
                if (col0 + n1 * G::Q + tid - bank >= prm.nbins) vmq &= ~(1u << n1);
            }
        }
        // The z = 0 slot has row_q == row_p and q == p bit for bit (H_0 is real), so its second
        // store rewrites the same value: no special case (MODE 1 reports the cell once: vq = 0).
        const unsigned qon = (MODE != 0 && row_q == row_p) ? 0u : ~0u;
        if constexpr (BANKS == 2) {
            // column 2 * bin + bank; the z = 0 slot's q row is its p row again (one bin off in bank 1): skipped
            float *bp = prm.plane + (size_t)row_p * prm.ncols + (2 * (col0 + tid) + bank);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + (2 * (col0 + tid - bank) + bank);
            emit_unit<L, false, MODE, 2>(prm, y, bp, bq, vm, row_q == row_p ? 0u : vmq);
        } else if constexpr (!INTERBIN) {
            float *bp = prm.plane + (size_t)row_p * prm.ncols + (col0 + tid);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + (col0 + tid);
            emit_unit<L, false, MODE, 1>(prm, y, bp, bq, vm, vmq & qon);
        } else {
            // lanes 0 and 31 post their y to the mailbox; lane 31's cells (power and half-bin) are
            // written one unit later by flush_edges, every other lane stores (P[n], P[n+1/2]) now
            float4 *eb = edges + par * (2 * G::W * 16) + (tm.lane == 0 ? G::W * 16 : 0) + tm.warp * 16;
            if (tm.lane == 31 || tm.lane == 0) {
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1)
                    eb[n1] = make_float4(y[n1].re.x, y[n1].re.y, y[n1].im.x, y[n1].im.y);
            }
            float *bp = prm.plane + (size_t)row_p * prm.ncols + 2 * (col0 + tid);
            float *bq = prm.plane + (size_t)row_q * prm.ncols + 2 * (col0 + tid);
            if (tm.lane == 31) vm = 0;
            emit_unit<L, true, MODE, 1>(prm, y, bp, bq, vm, vm & qon);
            pend.col0 = col0;
            pend.pair = row_p;
            pend.par = par;
            pend.on = true;
        }
        __syncwarp();
        if (++pair == prm.npairs) {
            pair = 0;
            ++seg;
        }
    }
    if (INTERBIN && pend.on) {
        __syncthreads();
        flush_edges<L, MODE>(prm, tm, edges, pend);
    }
}

#endif // __CUDACC__

} // namespace fdas
