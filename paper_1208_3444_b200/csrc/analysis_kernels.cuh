// analysis_kernels.cuh -- the two O(N) / O(k S^2) outputs the paper attaches to the hot path
// (NEXT rows f3, f4 of SURVEY 8f), on sm_100a:
//   * splat_kernel           : headless particle-count snapshot, the content of the paper's live display
//                              (App. A step 7) and of Fig. 1; reading G23
//   * trace_spectrum_kernel  : periodogram of each tracer's recorded velocity series, "its energy power
//                              spectrum"; reading G24
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace colatus {

// ---- f4: particle-count image ---------------------------------------------------------------------
// Orthographic projection along `axis`; (u, v) = the two other coordinates in cyclic order, w = depth.
// A particle is counted iff w0 <= w < w1 and 0 <= (u-u0)*su < W and 0 <= (v-v0)*sv < H, all in FP32
// with every operation rounded once (__fsub_rn / __fmul_rn: no FMA contraction, so the integer pixel
// decision is reproducible on any IEEE machine).  su = W/(u1-u0), sv = H/(v1-v0) come from the host
// (one IEEE float division each).  Counts are exact integers: red.global.add.u32, order-independent.
// HBM-bound: 16 B read per body; the image (W*H*4 B) normally sits in L2.  A warp first merges lanes
// that hit the same pixel (match.any) so that a dense clump costs one atomic per distinct pixel.
__global__ void __launch_bounds__(256)
splat_kernel(const float4 *__restrict__ pos_mass, int64_t n, int axis, float u0, float su, float v0, float sv,
             float w0, float w1, int width, int height, uint32_t *__restrict__ image) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int pixel = -1;
    if (i < n) {
        const float4 p = pos_mass[i];
        const float u = axis == 0 ? p.y : (axis == 1 ? p.z : p.x);
        const float v = axis == 0 ? p.z : (axis == 1 ? p.x : p.y);
        const float w = axis == 0 ? p.x : (axis == 1 ? p.y : p.z);
        const float tu = __fmul_rn(__fsub_rn(u, u0), su);
        const float tv = __fmul_rn(__fsub_rn(v, v0), sv);
        if (w >= w0 && w < w1 && tu >= 0.f && tu < (float)width && tv >= 0.f && tv < (float)height)
            pixel = (int)floorf(tv) * width + (int)floorf(tu);
    }
    const unsigned peers = __match_any_sync(0xffffffffu, pixel);
    if (pixel >= 0 && (int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(image + pixel, (uint32_t)__popc(peers));
}

// ---- f3: periodogram of the tracer velocity series ---------------------------------------------------
//   P_t[f] = (1/S) sum_{c=x,y,z} | sum_{s<S} v_{t,c}[s] exp(-2 pi i f s / S) |^2,   f = 0 .. S/2
// ring rows are float4 (vx, vy, vz, tag) [capacity][k]; step first_step + s lives in row
// (first_step + s) % capacity.  One thread per (tracer, frequency): threadIdx.x runs over tracers so the
// ring reads are coalesced and every lane of a warp shares the twiddle argument.  The phase index
// (f s) mod S is advanced exactly in integers; twiddles and sums are FP64 (the record is short: k S^2 / 2
// terms, 1.6e7 for the paper-shaped 64 tracers x 1000 steps), samples stay the FP32 values of the ring.
__global__ void __launch_bounds__(256)
trace_spectrum_kernel(const float4 *__restrict__ ring, int k, int capacity, int64_t first_step, int S,
                      double *__restrict__ out) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int f = blockIdx.y * blockDim.y + threadIdx.y;
    const int nf = S / 2 + 1;
    if (t >= k || f >= nf) return;
    double rx = 0.0, ix = 0.0, ry = 0.0, iy = 0.0, rz = 0.0, iz = 0.0;
    int phase = 0;                                      // (f * s) mod S
    int row = (int)(first_step % capacity);
    const double inv_S = 2.0 / (double)S;               // sincospi argument = 2 * phase / S
    for (int s = 0; s < S; ++s) {
        double sn, cs;
        sincospi((double)phase * inv_S, &sn, &cs);
        const float4 v = ring[(size_t)row * k + t];
        rx = fma((double)v.x, cs, rx);
        ix = fma(-(double)v.x, sn, ix);
        ry = fma((double)v.y, cs, ry);
        iy = fma(-(double)v.y, sn, iy);
        rz = fma((double)v.z, cs, rz);
        iz = fma(-(double)v.z, sn, iz);
        phase += f;
        if (phase >= S) phase -= S;
        if (++row == capacity) row = 0;
    }
    out[(size_t)t * nf + f] = (rx * rx + ix * ix + ry * ry + iy * iy + rz * rz + iz * iz) / (double)S;
}

}  // namespace colatus
