// Red-noise removal and block normalisation of the spectrum, the two steps of Fig. 2 between the real-to-complex
// transform and the correlations.
//
// "low frequency (red) noise is removed with the use of a local median filter ... the signal size is
// divided into blocks ... After a short step of normalization on the data of each block, the matched filtering is
// performed".  The paper gives neither formula; readings R19 / R20:
//
//     out[j] = A[j] / sqrt(stat_b),   b = j / block,
//     stat_b = median_{j in b} |A[j]|^2 / ln 2      (FDAS_WHITEN_MEDIAN: red-noise removal; exponential noise powers
//                                                    have median = mean ln 2, so the noise comes out at unit mean)
//     stat_b = mean_{j in b}   |A[j]|^2             (FDAS_WHITEN_MEAN: unit mean power per overlap-save block)
//
// blocks are consecutive runs of `block` bins from bin 0 (the last one shorter); a block with stat_b = 0 is copied.
//
// One CTA per block.  The powers go to shared memory as bit patterns (non-negative floats order like unsigned
// integers); the median is EXACT: a most-significant-byte-first radix selection (four 256-bin histogram passes for
// rank w/2, plus one counting pass for rank w/2 - 1 when the count is even) instead of a sort -- O(w) work, no data
// movement.  (Measured negatives: a second selection for the lower rank, 0.095 ms against 0.067 ms at 2^23 bins
// in blocks of 1024; electing one lane per equal digit with __match_any_sync before the atomicAdd, 0.172 ms.)  The
// mean is a double sum.  The scale is formed once per block in double and rounded to float; the block is then read a second time (an
// L1/L2 hit: a block is at most 64 KB) and written scaled, so in-place use is safe (a thread reads a bin before it
// writes it, and no CTA touches another block).  Roofline: HBM, 16 N bytes (8 N read, 8 N written).
#pragma once
#include <stdint.h>

namespace fdas {

constexpr int WHITEN_THREADS = 256;
constexpr int WHITEN_MIN_BLOCK = 32, WHITEN_MAX_BLOCK = 8192;

inline size_t whiten_smem_bytes(int block) { return (size_t)block * 4 + 256 * 4 + 2 * 4 + 8 + 8 * 8; }

#ifdef __CUDACC__

// k-th smallest (k = 0 .. n-1) of the n bit patterns sp[0..n), for the whole CTA.  hist: 256 counters, bc: 2 words.
__device__ __forceinline__ unsigned whiten_select(const unsigned *sp, int n, int k, unsigned *hist, unsigned *bc)
{
    unsigned prefix = 0, mask = 0;
    for (int shift = 24; shift >= 0; shift -= 8) {
        for (int i = threadIdx.x; i < 256; i += blockDim.x) hist[i] = 0;
        __syncthreads();
        for (int i = threadIdx.x; i < n; i += blockDim.x) {
            const unsigned v = sp[i];
            if ((v & mask) == prefix) atomicAdd(&hist[(v >> shift) & 255u], 1u);
        }
        __syncthreads();
        if (threadIdx.x < 32) {                          // the bucket that holds rank k among the matching values
            const int lane = threadIdx.x;
            unsigned c[8], s = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                c[j] = hist[8 * lane + j];
                s += c[j];
            }
            unsigned incl = s;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            unsigned below = incl - s;
            if ((unsigned)k >= below && (unsigned)k < incl) {        // exactly one lane
                int j = 0;
                for (; j < 7; ++j) {
                    if ((unsigned)k < below + c[j]) break;
                    below += c[j];
                }
                bc[0] = (unsigned)(8 * lane + j);
                bc[1] = below;
            }
        }
        __syncthreads();
        prefix |= bc[0] << shift;
        mask |= 0xffu << shift;
        k -= (int)bc[1];
    }
    return prefix;
}

__global__ void __launch_bounds__(WHITEN_THREADS) whiten_kernel(const float2 *in, float2 *out,   // may alias (in place)
                                                                long long nbins, int block, int statistic)
{
    extern __shared__ __align__(16) unsigned char whiten_smem[];
    unsigned *sp = reinterpret_cast<unsigned *>(whiten_smem);
    unsigned *hist = sp + block;
    unsigned *bc = hist + 256;
    double *red = reinterpret_cast<double *>(whiten_smem + (((size_t)block * 4 + 256 * 4 + 2 * 4 + 7) & ~(size_t)7));
    const long long start = (long long)blockIdx.x * block;
    const int w = (int)(nbins - start < (long long)block ? nbins - start : (long long)block);
    const float2 *a = in + start;
    double acc = 0.0;
    for (int i = threadIdx.x; i < w; i += blockDim.x) {
        const float2 v = a[i];
        const float p = fmaf(v.y, v.y, v.x * v.x);
        sp[i] = __float_as_uint(p);
        acc += (double)p;
    }
    double stat;
    if (statistic == 1) {                                 // mean power
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
        __syncthreads();
        stat = 0.0;
        for (int i = 0; i < WHITEN_THREADS / 32; ++i) stat += red[i];      // same order in every thread
        stat /= (double)w;
    } else {                                              // median power / ln 2
        __syncthreads();
        const unsigned hi = whiten_select(sp, w, w / 2, hist, bc);
        unsigned lo = hi;
        if (!(w & 1)) {
            // even count: rank w/2 - 1 is the largest value below `hi` if exactly w/2 values lie below it, else it
            // equals `hi` (a tie) -- one counting pass instead of a second selection
            __syncthreads();
            if (threadIdx.x == 0) bc[0] = bc[1] = 0;
            __syncthreads();
            unsigned cnt = 0, mx = 0;
            for (int i = threadIdx.x; i < w; i += blockDim.x) {
                const unsigned v = sp[i];
                if (v < hi) {
                    ++cnt;
                    mx = v > mx ? v : mx;
                }
            }
            cnt = __reduce_add_sync(0xffffffffu, cnt);
            mx = __reduce_max_sync(0xffffffffu, mx);
            if ((threadIdx.x & 31) == 0) {
                atomicAdd(&bc[0], cnt);
                atomicMax(&bc[1], mx);
            }
            __syncthreads();
            if (bc[0] == (unsigned)(w / 2)) lo = bc[1];
        }
        stat = 0.5 * ((double)__uint_as_float(lo) + (double)__uint_as_float(hi)) / 0.693147180559945309417;
    }
    const float s = stat > 0.0 ? (float)(1.0 / sqrt(stat)) : 1.0f;
    for (int i = threadIdx.x; i < w; i += blockDim.x) {
        const float2 v = a[i];
        out[start + i] = make_float2(v.x * s, v.y * s);
    }
}

#endif // __CUDACC__

} // namespace fdas
