// integrate_kernels.cuh -- eqs. (3)-(5) of arXiv 1208.3444 and the tracer record.
//
//   x^{n+1/2} = x^n + (tau/2) v^n                                                     (3)  drift_kernel
//   v^{n+1}   = v^n (1-H tau)/(1+H tau) + F tau/(a^3 (1+H tau))                       (4)  kick_drift_kernel
//   x^{n+1}   = x^{n+1/2} + (tau/2) v^{n+1}                                           (5)  (same kernel)
//
// The coefficients d1 = tau/2, cv = (1-H tau)/(1+H tau), ck = tau/(a^3 (1+H tau)), d2 = tau/2 are
// formed in double on the host.  Elementwise, HBM-bound: one float4 per array per body, coalesced.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "force_kernels.cuh"

namespace colatus {

// The drift kernels update x, y, z only and never store .w, so that the mass a neighbouring thread may be reading
// (body 0's, for the equal-mass detection) is not written concurrently.
__device__ __forceinline__ void store_xyz(float4 *dst, const float4 &p) {
    *reinterpret_cast<float2 *>(dst) = make_float2(p.x, p.y);
    reinterpret_cast<float *>(dst)[2] = p.z;
}

// eq. (3): x += d v   (mass in .w untouched)
__global__ void __launch_bounds__(256) drift_kernel(float4 *__restrict__ pos_mass, const float4 *__restrict__ vel,
                                                    int64_t begin, int64_t count, float d) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    float4 p = pos_mass[begin + i];
    const float4 v = vel[begin + i];
    p.x = fmaf(d, v.x, p.x);
    p.y = fmaf(d, v.y, p.y);
    p.z = fmaf(d, v.z, p.z);
    pos_mass[begin + i] = p;
}

// eqs. (4)+(5) fused, plus the tracer record: acc is indexed from 0 for the
// target range.  trace_slot[k] >= 0 marks particle k as tracer number trace_slot[k]; its v^{n+1}
// goes to ring_row[slot] = (vx, vy, vz, tag).
template <bool TRACE>
__global__ void __launch_bounds__(256)
kick_drift_kernel(float4 *__restrict__ pos_mass, float4 *__restrict__ vel, const float4 *__restrict__ acc,
                  int64_t begin, int64_t count, float cv, float ck, float d2,
                  const int32_t *__restrict__ trace_slot, float4 *__restrict__ ring_row, float tag) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    float4 p = pos_mass[begin + i];
    float4 v = vel[begin + i];
    const float4 f = acc[i];
    v.x = fmaf(ck, f.x, cv * v.x);
    v.y = fmaf(ck, f.y, cv * v.y);
    v.z = fmaf(ck, f.z, cv * v.z);
    p.x = fmaf(d2, v.x, p.x);
    p.y = fmaf(d2, v.y, p.y);
    p.z = fmaf(d2, v.z, p.z);
    vel[begin + i] = v;
    pos_mass[begin + i] = p;
    if (TRACE) {
        const int32_t s = trace_slot[begin + i];
        if (s >= 0) ring_row[s] = make_float4(v.x, v.y, v.z, tag);
    }
}

// ---- table-driven variants for colatus_run (CUDA-graph replay of a launch-bound step loop) ----------------
// The per-step coefficients live in a device table; a device counter selects the row, so the five
// kernels of a step have step-independent arguments and ONE captured graph is replayed every step.
//   ctr[0] = step index the next drift uses;  ctr[1] = step index the kick-drift uses.
// drift copies ctr[0] into ctr[1] (nobody reads ctr[1] while drift runs); kick-drift writes
// ctr[0] = step + 1 (nobody reads ctr[0] while it runs).  Same arithmetic as the scalar kernels.
struct StepCoef {
    float d1, cv, ck, d2, tag;
    int ring_row;       // (step % capacity) of this step's tracer row
    float d1_next;      // first half-drift coefficient of the step after this one (two-kernel loop below)
    int has_next;       // 0 for the last step of a colatus_run call; 32 B per row
};

__global__ void __launch_bounds__(256)
drift_table_kernel(float4 *__restrict__ pos_mass, const float4 *__restrict__ vel, int64_t begin, int64_t count,
                   const StepCoef *__restrict__ table, int *__restrict__ ctr) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int s = ctr[0];
    if (i == 0) ctr[1] = s;
    if (i >= count) return;
    const float d = table[s].d1;
    float4 p = pos_mass[begin + i];
    const float4 v = vel[begin + i];
    p.x = fmaf(d, v.x, p.x);
    p.y = fmaf(d, v.y, p.y);
    p.z = fmaf(d, v.z, p.z);
    pos_mass[begin + i] = p;
}

template <bool TRACE>
__global__ void __launch_bounds__(256)
kick_drift_table_kernel(float4 *__restrict__ pos_mass, float4 *__restrict__ vel, const float4 *__restrict__ acc,
                        int64_t begin, int64_t count, const StepCoef *__restrict__ table, int *__restrict__ ctr,
                        const int32_t *__restrict__ trace_slot, float4 *__restrict__ ring, int trace_k) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int s = ctr[1];
    if (i == 0) ctr[0] = s + 1;
    if (i >= count) return;
    const StepCoef c = table[s];
    float4 p = pos_mass[begin + i];
    float4 v = vel[begin + i];
    const float4 f = acc[i];
    v.x = fmaf(c.ck, f.x, c.cv * v.x);
    v.y = fmaf(c.ck, f.y, c.cv * v.y);
    v.z = fmaf(c.ck, f.z, c.cv * v.z);
    p.x = fmaf(c.d2, v.x, p.x);
    p.y = fmaf(c.d2, v.y, p.y);
    p.z = fmaf(c.d2, v.z, p.z);
    vel[begin + i] = v;
    pos_mass[begin + i] = p;
    if (TRACE) {
        const int32_t t = trace_slot[begin + i];
        if (t >= 0) ring[(size_t)c.ring_row * trace_k + t] = make_float4(v.x, v.y, v.z, c.tag);
    }
}

// ---- fused step kernels (whole-range steps without external terms) ----------------------------------------
// A leapfrog step is launch-bound at small N, so the two O(N) passes next to the force kernel are folded
// into their neighbours: drift + staging (eq. (3) and the padded source copy the force kernel reads), and
// partial-sum reduction + kick + drift (+ tracer record) (eqs. (4), (5)).  Three launches per step instead of
// five; the arithmetic, statement for statement, is that of drift_kernel / stage_sources_kernel /
// reduce_partials_kernel / kick_drift_kernel, so the results are bitwise the same.
// Coefficients come from the scalar arguments, or -- table != nullptr -- from the device table row the step
// counters select (see the table-driven variants above).
struct StepSrc {
    const StepCoef *table;   // nullptr: use the scalars below
    int *ctr;
    float d1, cv, ck, d2, tag;
    int ring_row;
};

__global__ void __launch_bounds__(256)
drift_stage_kernel(float4 *__restrict__ pos_mass, const float4 *__restrict__ vel, int64_t n, int64_t n_pad,
                   float4 *__restrict__ staged, int *__restrict__ mass_flag, int generation, StepSrc src) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    float d = src.d1;
    if (src.table) {
        const int s = src.ctr[0];
        if (j == 0) src.ctr[1] = s;
        d = src.table[s].d1;
    }
    if (j >= n_pad) return;
    if (j < n) {
        const float m0 = pos_mass[0].w;          // body 0's mass: no thread of this kernel stores a .w (store_xyz)
        float4 p = pos_mass[j];
        const float4 v = vel[j];
        p.x = fmaf(d, v.x, p.x);
        p.y = fmaf(d, v.y, p.y);
        p.z = fmaf(d, v.z, p.z);
        store_xyz(pos_mass + j, p);
        staged[j] = p;
        if (p.w != m0) mass_flag[0] = generation;
    } else {
        staged[j] = make_float4(PAD_FAR, PAD_FAR, PAD_FAR, 0.f);
    }
}

template <bool TRACE>
__global__ void __launch_bounds__(256)
reduce_kick_drift_kernel(float4 *__restrict__ pos_mass, float4 *__restrict__ vel, float4 *__restrict__ acc,
                         const float4 *__restrict__ partial, int64_t stride, int splits, int64_t n, float G,
                         StepSrc src, const int32_t *__restrict__ trace_slot, float4 *__restrict__ ring,
                         int trace_k) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    float cv = src.cv, ck = src.ck, d2 = src.d2, tag = src.tag;
    int ring_row = src.ring_row;
    if (src.table) {
        const int s = src.ctr[1];
        if (i == 0) src.ctr[0] = s + 1;
        const StepCoef c = src.table[s];
        cv = c.cv; ck = c.ck; d2 = c.d2; tag = c.tag; ring_row = c.ring_row;
    }
    if (i >= n) return;
    const float4 s4 = sum_partials(partial, stride, splits, i);
    const float4 f = make_float4(s4.x * G, s4.y * G, s4.z * G, 0.f);
    acc[i] = f;                                   // the caller's acc buffer still receives F
    float4 p = pos_mass[i];
    float4 v = vel[i];
    v.x = fmaf(ck, f.x, cv * v.x);
    v.y = fmaf(ck, f.y, cv * v.y);
    v.z = fmaf(ck, f.z, cv * v.z);
    p.x = fmaf(d2, v.x, p.x);
    p.y = fmaf(d2, v.y, p.y);
    p.z = fmaf(d2, v.z, p.z);
    vel[i] = v;
    pos_mass[i] = p;
    if (TRACE) {
        const int32_t t = trace_slot[i];
        if (t >= 0) ring[(size_t)ring_row * trace_k + t] = make_float4(v.x, v.y, v.z, tag);
    }
}

// ---- two-kernel step loop of colatus_run ------------------------------------------------------------------
// Inside a run the tail of step s (partial sums, kick, drift, tracer record) and the head of step s+1 (first
// half drift, staging, equal-mass detection) are consecutive elementwise passes over the same bodies, so they
// share a kernel: a step is then TWO launches, force_kernel + step_tail_head_kernel (the very first head of a
// run is one drift_stage_kernel).  Statement for statement the arithmetic is that of reduce_kick_drift_kernel
// followed by drift_stage_kernel -- two separately rounded drifts, not one merged one -- so the bits equal
// those of colatus_step.  Row ctr[1] of the table holds the step's coefficients plus d1 of the next step;
// has_next = 0 on the last step of the run leaves x^{n+1} in place.  splits = 0: acc already holds G * sum.
// The grid covers n_pad (the padding of the staged array is rewritten with far-away massless bodies).
template <bool TRACE>
__global__ void __launch_bounds__(256)
step_tail_head_kernel(float4 *__restrict__ pos_mass, float4 *__restrict__ vel, float4 *__restrict__ acc,
                      const float4 *__restrict__ partial, int64_t stride, int splits, int64_t n, int64_t n_pad,
                      float G, const StepCoef *__restrict__ table, int *__restrict__ ctr,
                      const int32_t *__restrict__ trace_slot, float4 *__restrict__ ring, int trace_k,
                      float4 *__restrict__ staged, int *__restrict__ mass_flag, int generation) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    // Launched as a programmatic dependent of the force kernel: everything the force kernel does not write --
    // positions, velocities, the tracer map -- is loaded BEFORE the wait, so these loads overlap the end of the
    // force kernel; only the step counter, the partial sums and acc wait for it.
    float4 p = make_float4(0.f, 0.f, 0.f, 0.f), v = p;
    float m0 = 0.f;
    int32_t tslot = -1;
    if (i < n) {
        p = pos_mass[i];
        v = vel[i];
        m0 = pos_mass[0].w;                       // no thread of this kernel stores a .w (store_xyz)
        if (TRACE) tslot = trace_slot[i];
    }
    griddep_wait();
    griddep_launch_dependents();
    const int s = ctr[1];                        // set by the force kernel of this step (ctr[1] = ctr[0])
    if (i == 0) ctr[0] = s + 1;
    if (i >= n_pad) return;
    float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
    if (i < n) {                                 // issued together with the counter load: independent of it
        if (splits > 0) {
            const float4 s4 = sum_partials(partial, stride, splits, i);
            f = make_float4(s4.x * G, s4.y * G, s4.z * G, 0.f);
            acc[i] = f;                           // the caller's acc buffer still receives F
        } else {
            f = acc[i];
        }
    }
    const StepCoef c = table[s];
    if (i >= n) {
        if (c.has_next) staged[i] = make_float4(PAD_FAR, PAD_FAR, PAD_FAR, 0.f);
        return;
    }
    v.x = fmaf(c.ck, f.x, c.cv * v.x);
    v.y = fmaf(c.ck, f.y, c.cv * v.y);
    v.z = fmaf(c.ck, f.z, c.cv * v.z);
    p.x = fmaf(c.d2, v.x, p.x);
    p.y = fmaf(c.d2, v.y, p.y);
    p.z = fmaf(c.d2, v.z, p.z);
    vel[i] = v;
    if (TRACE) {
        if (tslot >= 0) ring[(size_t)c.ring_row * trace_k + tslot] = make_float4(v.x, v.y, v.z, c.tag);
    }
    if (c.has_next) {                             // head of the next step: eq. (3) and the staged copy
        p.x = fmaf(c.d1_next, v.x, p.x);
        p.y = fmaf(c.d1_next, v.y, p.y);
        p.z = fmaf(c.d1_next, v.z, p.z);
        staged[i] = p;
        if (p.w != m0) mass_flag[0] = generation;
    }
    store_xyz(pos_mass + i, p);
}

// External terms added to the force of eq. (1) for the target range (acc indexed from 0):
//   eq. (10), PAPER.md:93 (reading G21):  F_k += S (x_psi - x_k) / (|x_k - x_psi|^2 + eps^2)^{3/2}
//   background (reading G22):             F_k += B (x_k - centre),  B = (4 pi / 3) G rho_bar (host, double)
// O(n), IEEE division and square root (not on the hot path); acc.w is left alone.
__global__ void __launch_bounds__(256)
external_field_kernel(const float4 *__restrict__ pos_mass, int64_t begin, int64_t count, float4 *__restrict__ acc,
                      float S, float px, float py, float pz, float eps2, float B, float cx, float cy, float cz) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const float4 p = pos_mass[begin + i];
    float4 f = acc[i];
    if (S != 0.f) {
        const float dx = px - p.x, dy = py - p.y, dz = pz - p.z;
        const float s = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, eps2)));
        const float w = S / (s * sqrtf(s));
        f.x = fmaf(w, dx, f.x);
        f.y = fmaf(w, dy, f.y);
        f.z = fmaf(w, dz, f.z);
    }
    if (B != 0.f) {
        f.x = fmaf(B, p.x - cx, f.x);
        f.y = fmaf(B, p.y - cy, f.y);
        f.z = fmaf(B, p.z - cz, f.z);
    }
    acc[i] = f;
}

// tracer slot map: slot[k] = t if idx[t] == k else -1
__global__ void __launch_bounds__(256) trace_fill_kernel(int32_t *__restrict__ slot, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) slot[i] = -1;
}
__global__ void __launch_bounds__(256)
trace_scatter_kernel(int32_t *__restrict__ slot, int64_t n, const int32_t *__restrict__ idx, int k) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < k) {
        const int32_t j = idx[t];
        if (j >= 0 && (int64_t)j < n) slot[j] = t;
    }
}

// ---- diagnostics (eq. (7)): FP64 accumulation, fixed order ---------------------------
// per-block partial q[0..8] = sum m, sum m vx, sum m vy, sum m vz, sum m v^2, sum m x, sum m y, sum m z,
// sum m phi (phi = acc.w of a potential pass, or 0).
constexpr int DIAG_Q = 9;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__global__ void __launch_bounds__(256) diagnostics_partial_kernel(const float4 *__restrict__ pos_mass,
                                                                  const float4 *__restrict__ vel,
                                                                  const float4 *__restrict__ phi_w, int64_t n,
                                                                  double *__restrict__ partial) {
    double q[DIAG_Q];
#pragma unroll
    for (int c = 0; c < DIAG_Q; ++c) q[c] = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float4 p = pos_mass[i];
        const float4 v = vel[i];
        const double m = p.w;
        q[0] += m;
        q[1] += m * v.x;
        q[2] += m * v.y;
        q[3] += m * v.z;
        q[4] += m * ((double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z);
        q[5] += m * p.x;
        q[6] += m * p.y;
        q[7] += m * p.z;
        if (phi_w) q[8] += m * phi_w[i].w;
    }
    __shared__ double sh[8][DIAG_Q];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int c = 0; c < DIAG_Q; ++c) {
        const double s = warp_sum(q[c]);
        if (lane == 0) sh[warp][c] = s;
    }
    __syncthreads();
    if (threadIdx.x < DIAG_Q) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += sh[w][threadIdx.x];
        partial[(size_t)blockIdx.x * DIAG_Q + threadIdx.x] = s;
    }
}

// One warp per quantity: lane l adds partials l, l+32, ... in order, then a fixed xor-shuffle tree -- the
// summation order depends only on `blocks`, so the result is reproducible.  Launch with DIAG_Q warps.
__global__ void __launch_bounds__(DIAG_Q * 32)
diagnostics_final_kernel(const double *__restrict__ partial, int blocks, double *__restrict__ out) {
    const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double s = 0.0;
    for (int b = lane; b < blocks; b += 32) s += partial[(size_t)b * DIAG_Q + c];
    s = warp_sum(s);
    if (lane == 0) out[c] = s;
}

}  // namespace colatus
