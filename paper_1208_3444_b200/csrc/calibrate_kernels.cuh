// calibrate_kernels.cuh -- register-only FP32 FMA loops that measure the denominator of the "alu" roofline
// (DESIGN.md 6.1): MEASURED_PEAKS.json carries HBM and bf16 figures but no FP32 one, so the library can
// time the plain-ALU peak itself on the device it runs on.  PACKED = 0: scalar FFMA; 1: FFMA2 (f32x2).
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
//   0: 12 FFMA2 (two shared operands)            3: 12 FFMA2 with three distinct 64-bit register operands
//   1: 12 FFMA2 + 2 MUFU.RSQ                      4: 12 FFMA2 + 1 LDS.128 (broadcast address)
//   2: 12 FFMA2 + 2 IADD                          5: 24 scalar FFMA + 2 MUFU.RSQ
constexpr int PROBE_GROUPS = 2048;   // groups per warp

template <int MODE>
__global__ void __launch_bounds__(CAL_THREADS) pipe_probe_kernel(float a, float b, float *__restrict__ sink) {
    __shared__ float4 tile[64];
    if (threadIdx.x < 64) tile[threadIdx.x] = make_float4(a, b, a, b);
    __syncthreads();
    u64 x[CAL_CHAINS], y[CAL_CHAINS], z[CAL_CHAINS];
    float xs[2 * CAL_CHAINS];
    const u64 A = pack2(a, a), Bv = pack2(b, b);
#pragma unroll
    for (int c = 0; c < CAL_CHAINS; ++c) {
        x[c] = pack2((float)threadIdx.x + c, (float)blockIdx.x - c);
        y[c] = pack2(b * (c + 1), b * (c + 2));
        z[c] = pack2(a - 1e-3f * c, a - 2e-3f * c);
        xs[2 * c] = (float)threadIdx.x + c;
        xs[2 * c + 1] = (float)blockIdx.x - c;
    }
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
            } else {
#pragma unroll
                for (int c = 0; c < 12; ++c) {
                    const int q = c % CAL_CHAINS;
                    x[q] = MODE == 3 ? fma2(x[q], z[q], y[q]) : fma2(x[q], A, Bv);
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
                asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                             : "=f"(v0), "=f"(v1), "=f"(v2), "=f"(v3)
                             : "r"(tile_addr + ((it & 31) << 4)));
            }
        }
    }
    float s = r0 + r1 + (float)(k0 ^ k1);
#pragma unroll
    for (int c = 0; c < CAL_CHAINS; ++c) {
        float lo, hi;
        unpack2(x[c], lo, hi);
        s += lo + hi + xs[2 * c] + xs[2 * c + 1];
    }
    if (s == 123456.789f) sink[0] = s;
}

}  // namespace colatus
