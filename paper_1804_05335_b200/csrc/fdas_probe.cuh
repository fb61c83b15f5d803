// Instruction-cost probes behind the "what bounds the kernel" argument of DESIGN.md section 6:
// cycles per warp instruction of the packed-FP32 and shared-memory instructions the fused kernel
// is made of, and of a unit-shaped mix of the two.  Not on the hot path; fdas_probe_pipes() runs
// them on one CTA per SM with 8 warps (two per SM sub-partition, like the fused kernel).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fdas {

enum ProbeMode { PROBE_FFMA = 0, PROBE_FADD2, PROBE_FFMA2, PROBE_FFMA2_3PAIR, PROBE_FMUL2, PROBE_LDS_STS64,
                 PROBE_SHFL, PROBE_MIX, PROBE_COUNT };

// One round = 16 "slots"; FP modes issue FPI instructions per slot, memory modes one LDS.64 and
// one STS.64 (or four SHFL) per slot; PROBE_MIX = per round 16 LDS.64 + 16 STS.64 + 128 packed ops
// (the fused kernel's unit: 128 LDS/STS.64 + 548 packed ops + 93 scalar).
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

// Tensor-memory probe (could TMEM hold the thread-private X^ / twiddle registers?):
// cycles per warp-wide tcgen05.ld / tcgen05.st of 32 columns (32x32b.x32: one 32-bit word per lane and column,
// lane-private like a register), 8 warps per SM, each on its own lane quadrant / column block.
// mode 0: load + wait::ld per instruction (latency-exposed), 1: four loads per wait, 2: four stores per wait.
__global__ void __launch_bounds__(256, 1) tmem_probe_kernel(float *out, int iters, int mode)
{
    __shared__ uint32_t taddr_sm;
    const int warp = threadIdx.x >> 5;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;"
                     ::"r"((uint32_t)__cvta_generic_to_shared(&taddr_sm)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t base = taddr_sm;
    const uint32_t addr = base + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(warp >> 2) * 32u;
    uint32_t r[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) r[i] = threadIdx.x * 32u + i;
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(addr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31]) : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    uint32_t acc = 0;
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (mode == 2) {
                asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(addr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31]) : "memory");
            } else {
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31]) : "r"(addr) : "memory");
                if (mode == 0) {
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    acc ^= r[k];
                }
            }
        }
        if (mode == 2) asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        else asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        acc += r[0];
    }
    const long long t1 = clock64();
    bool ok = true;                                   // what was stored is what comes back
#pragma unroll
    for (int i = 0; i < 32; ++i) ok = ok && (r[i] == threadIdx.x * 32u + i);
    if (acc == 0x12345u) out[0] = 1.f;
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        out[1] = (float)(t1 - t0);
        out[2] = ok ? 1.f : 0.f;
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" ::"r"(base) : "memory");
}

} // namespace fdas
