// probe_kernels.cuh -- kernels of libcolatus_probe (include/colatus_probe.h), NOT of the product library.
// Register-only FP32 FMA loops that measure the denominator of the "alu" roofline:
// MEASURED_PEAKS.json carries HBM and bf16 figures but no FP32 one, so the plain-ALU peak is timed on the
// device itself.  PACKED = 0: scalar FFMA; 1: FFMA2 (f32x2).
// Each thread runs CHAINS independent dependent chains x = x * a + b, so the pipe is limited by issue,
// not latency; 2 flop per lane-FMA.  The result is stored only if it is NaN-like, which never happens
// for the chosen constants, but keeps the loop alive.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "force_kernels.cuh"

namespace colatus {

constexpr int CAL_THREADS = 256;
constexpr int CAL_CHAINS = 8;
constexpr int CAL_ITERS = 4096;
constexpr int CAL_UNROLL = 8;

template <int PACKED>
__global__ void __launch_bounds__(CAL_THREADS) calibrate_fma_kernel(float a, float b, float *__restrict__ sink) {
    if (PACKED) {
        u64 x[CAL_CHAINS];
        const u64 A = pack2(a, a), Bv = pack2(b, b);
#pragma unroll
        for (int c = 0; c < CAL_CHAINS; ++c) x[c] = pack2((float)threadIdx.x + c, (float)blockIdx.x - c);
#pragma unroll 1
        for (int it = 0; it < CAL_ITERS / CAL_UNROLL; ++it) {
#pragma unroll
            for (int u = 0; u < CAL_UNROLL; ++u)
#pragma unroll
                for (int c = 0; c < CAL_CHAINS; ++c) x[c] = fma2(x[c], A, Bv);
        }
        float s = 0.f;
#pragma unroll
        for (int c = 0; c < CAL_CHAINS; ++c) {
            float lo, hi;
            unpack2(x[c], lo, hi);
            s += lo + hi;
        }
        if (s == 123456.789f) sink[0] = s;
    } else {
        float x[2 * CAL_CHAINS];
#pragma unroll
        for (int c = 0; c < 2 * CAL_CHAINS; ++c) x[c] = (float)threadIdx.x + c - (float)blockIdx.x;
#pragma unroll 1
        for (int it = 0; it < CAL_ITERS / CAL_UNROLL; ++it) {
#pragma unroll
            for (int u = 0; u < CAL_UNROLL; ++u)
#pragma unroll
                for (int c = 0; c < 2 * CAL_CHAINS; ++c) x[c] = fmaf(x[c], a, b);
        }
        float s = 0.f;
#pragma unroll
        for (int c = 0; c < 2 * CAL_CHAINS; ++c) s += x[c];
        if (s == 123456.789f) sink[0] = s;
    }
}

// ---- issue-rule probes -------------------------------------------------------------------
// Register-only loops whose body is one "group" of 12 packed FP32 ops (the FP work of one packed
// pair-interaction) plus, per MODE, the extra instructions whose cost next to a saturated FMA pipe is in
// question.  The caller converts the launch time into SMSP cycles per group.
//   0: 12 FFMA2 x = x*A + B (two loop-constant operands)
//   1: 0 + 2 MUFU.RSQ                              2: 0 + 2 IADD
//   3: 12 accumulates a[t][c] = w[t]*d[t][c] + a[t][c], t-major: triples that share w (three distinct 64-bit
//      register operands each; the operand-reuse cache can hold w for the 2nd and 3rd of a triple)
//   4: 0 + 1 LDS.128 (broadcast address)           5: 24 scalar FFMA + 2 MUFU.RSQ
//   6: the accumulates of 3, c-major: w changes every instruction, no operand reuse possible
//   7: 0 + 6 DFMA (does the FP64 pipe run next to a saturated FP32 pipe?)
constexpr int PROBE_GROUPS = 2048;   // groups per warp

template <int MODE>
__global__ void __launch_bounds__(CAL_THREADS) pipe_probe_kernel(float a, float b, float *__restrict__ sink) {
    __shared__ float4 tile[64];
    if (threadIdx.x < 64) tile[threadIdx.x] = make_float4(a, b, a, b);
    __syncthreads();
    u64 w[4], d[4][3], acc[4][3];
    float xs[2 * CAL_CHAINS];
    double y[6];
    const u64 A = pack2(a, a), Bv = pack2(b, b);
    const double da = a, db = b;
#pragma unroll
    for (int c = 0; c < CAL_CHAINS; ++c) {
        xs[2 * c] = (float)threadIdx.x + c;
        xs[2 * c + 1] = (float)blockIdx.x - c;
    }
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        w[t] = pack2(a * (t + 1) * 1e-3f, b * (t + 2) * 1e-3f);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            d[t][c] = pack2(a + 0.01f * (t * 3 + c) + threadIdx.x * 1e-6f, b - 0.02f * (t * 3 + c));
            acc[t][c] = pack2((float)threadIdx.x, (float)blockIdx.x + c + t);
        }
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) y[c] = (double)threadIdx.x + c;
    float r0 = 1.5f + threadIdx.x, r1 = 2.5f + threadIdx.x;
    int k0 = threadIdx.x, k1 = blockIdx.x | 1;
    const uint32_t tile_addr = smem_u32(tile);
#pragma unroll 1
    for (int it = 0; it < PROBE_GROUPS / 2; ++it) {
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (MODE == 5) {
#pragma unroll
                for (int c = 0; c < 24; ++c) xs[c % (2 * CAL_CHAINS)] = fmaf(xs[c % (2 * CAL_CHAINS)], a, b);
            } else if (MODE == 3) {
#pragma unroll
                for (int t = 0; t < 4; ++t)
#pragma unroll
                    for (int c = 0; c < 3; ++c) acc[t][c] = fma2(w[t], d[t][c], acc[t][c]);
            } else if (MODE == 6) {
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int t = 0; t < 4; ++t) acc[t][c] = fma2(w[t], d[t][c], acc[t][c]);
            } else {
#pragma unroll
                for (int c = 0; c < 12; ++c) {                 // 12 independent chains
                    acc[c / 3][c % 3] = fma2(acc[c / 3][c % 3], A, Bv);
                    if (MODE == 7 && c < 6) y[c] = fma(y[c], da, db);
                }
            }
            if (MODE == 1 || MODE == 5) {
                r0 = rsqrt_approx(r0);
                r1 = rsqrt_approx(r1);
            }
            if (MODE == 2) {
                asm volatile("add.s32 %0, %0, %1;" : "+r"(k0) : "r"(k1));
                asm volatile("add.s32 %0, %0, %1;" : "+r"(k1) : "r"(k0));
            }
            if (MODE == 4) {
                float v0, v1, v2, v3;
                asm volatile("ld.volatile.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                             : "=f"(v0), "=f"(v1), "=f"(v2), "=f"(v3)
                             : "r"(tile_addr + ((it & 31) << 4)));
            }
        }
    }
    float s = r0 + r1 + (float)(k0 ^ k1);
#pragma unroll
    for (int c = 0; c < 2 * CAL_CHAINS; ++c) s += xs[c];
#pragma unroll
    for (int t = 0; t < 4; ++t)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            float lo, hi;
            unpack2(acc[t][c], lo, hi);
            s += lo + hi;
        }
#pragma unroll
    for (int c = 0; c < 6; ++c) s += (float)y[c];
    if (s == 123456.789f) sink[0] = s;
}

}  // namespace colatus
