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

}  // namespace colatus
