// Instruction-cost probes behind the "what bounds the kernel" argument of DESIGN.md section 6:
// cycles per warp instruction of the packed-FP32 and shared-memory instructions the fused kernel
// is made of, and of a unit-shaped mix of the two.  Not on the hot path; fdas_probe_pipes() runs
// them on one CTA per SM with 8 warps (two per SM sub-partition, like the fused kernel).
#pragma once
#include <cuda_runtime.h>

namespace fdas {

enum ProbeMode { PROBE_FFMA = 0, PROBE_FADD2, PROBE_FFMA2, PROBE_FFMA2_3PAIR, PROBE_FMUL2, PROBE_LDS_STS64,
                 PROBE_SHFL, PROBE_MIX, PROBE_COUNT };

// One round = 16 "slots"; FP modes issue FPI instructions per slot, memory modes one LDS.64 and
// one STS.64 (or four SHFL) per slot; PROBE_MIX = per round 16 LDS.64 + 16 STS.64 + 128 packed ops
// (the fused kernel's unit: 255 LDS/STS.64 + 548 packed ops + 93 scalar).
template <int MODE>
__global__ void __launch_bounds__(256, 1) probe_kernel(float *out, int iters, float s0, float s1)
{
    extern __shared__ float2 probe_sm[];
    const int tid = threadIdx.x, nt = blockDim.x;
    float2 a[16], b[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        a[i] = make_float2(tid + i, i * 0.5f);
        b[i] = make_float2(i + 1.f, tid * 0.25f + i);
    }
    for (int i = tid; i < 16 * nt; i += nt) probe_sm[i] = make_float2(i, -i);
    __syncthreads();
    const float2 c0 = make_float2(s0, s0);
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        if (MODE == PROBE_LDS_STS64 || MODE == PROBE_MIX) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                const float2 v = probe_sm[i * nt + tid];
                a[i].x += v.x;
                a[i].y += v.y;
            }
        }
        constexpr int REP = (MODE == PROBE_MIX) ? 4 : (MODE == PROBE_LDS_STS64 || MODE == PROBE_SHFL) ? 0 : 8;
#pragma unroll
        for (int r = 0; r < REP; ++r) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                if (MODE == PROBE_FFMA) { a[i].x = fmaf(a[i].x, s0, b[i].x); a[i].y = fmaf(a[i].y, s1, b[i].y); }
                if (MODE == PROBE_FADD2) a[i] = __fadd2_rn(a[i], b[i]);
                if (MODE == PROBE_FFMA2) a[i] = __ffma2_rn(a[i], c0, b[i]);
                if (MODE == PROBE_FFMA2_3PAIR) a[i] = __ffma2_rn(a[i], b[(i + 1) & 15], b[i]);
                if (MODE == PROBE_FMUL2) a[i] = __fmul2_rn(a[i], c0);
                if (MODE == PROBE_MIX) { a[i] = __fadd2_rn(a[i], b[i]); b[i] = __ffma2_rn(b[i], c0, a[(i + 3) & 15]); }
            }
        }
        if (MODE == PROBE_SHFL) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                a[i].x += __shfl_xor_sync(0xffffffffu, a[i].y, 4);
                a[i].y += __shfl_xor_sync(0xffffffffu, b[i].x, 8);
                b[i].x += __shfl_xor_sync(0xffffffffu, b[i].y, 16);
                b[i].y += __shfl_down_sync(0xffffffffu, a[i].x, 1);
            }
        }
        if (MODE == PROBE_LDS_STS64 || MODE == PROBE_MIX) {
#pragma unroll
            for (int i = 0; i < 16; ++i) probe_sm[i * nt + tid] = a[i];
        }
    }
    const long long t1 = clock64();
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) acc += a[i].x + a[i].y + b[i].x + b[i].y;
    if (acc == 123.456f) out[0] = acc;
    if (threadIdx.x == 0 && blockIdx.x == 0) out[1] = (float)(t1 - t0);
}

// warp instructions of the probed kind per round and thread
constexpr int probe_instr_per_round(int mode)
{
    return mode == PROBE_FFMA ? 8 * 16 * 2
         : mode == PROBE_LDS_STS64 ? 32
         : mode == PROBE_SHFL ? 64
         : mode == PROBE_MIX ? 1      // reported per round (16 LDS.64 + 16 STS.64 + 128 packed)
         : 8 * 16;
}

} // namespace fdas
