// force_kernels.cuh -- eq. (1) of arXiv 1208.3444 on sm_100a.
//
//   F_k = G * sum_{j != k} m_j (x_j - x_k) / (|x_j - x_k|^2 + eps^2)^{3/2}
//
// Design:
//   * repack kernel  : float4 (x,y,z,m)[n] -> source PAIRS (x0,x1,y0,y1)(z0,z1,m0,m1), zero-mass
//                      padding, so one 64-bit register holds the same coordinate of two sources;
//   * force kernel   : targets in registers (I per thread), source tiles staged in shared memory
//                      by 1-D bulk async copies (cp.async.bulk + mbarrier ring) and read as
//                      warp-broadcast LDS.128; arithmetic in packed FP32 (fma/add/mul.rn.f32x2 ->
//                      FFMA2/FADD2/FMUL2: two interactions per issue slot), rsqrt.approx on the
//                      MUFU pipe; accumulators flushed once per tile (blocked summation);
//   * the (target-tile x source-split) grid is sized to the machine, each split writes a
//     partial sum, and a fixed-order reduce kernel adds the partials and applies G.
// The self term needs no branch: d = 0 gives w*d = 0 exactly because eps^2 > 0 (reading G4).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace colatus {

typedef unsigned long long u64;

// ---- packed FP32 helpers (sm_100+) -----------------------------------------------------------
__device__ __forceinline__ u64 pack2(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(u64 v, float &lo, float &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- mbarrier / bulk-copy helpers ---------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
__device__ __forceinline__ void bulk_copy_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---- repack: AoS float4 -> source pairs -----------------------------------------------------------
// packed[2p]   = (x_{2p}, x_{2p+1}, y_{2p}, y_{2p+1})
// packed[2p+1] = (z_{2p}, z_{2p+1}, m_{2p}, m_{2p+1})        for p in [0, n_pad/2)
// Sources j >= n are padding: position 0, mass 0 (contribute exactly 0 to F and to phi).
__global__ void __launch_bounds__(256) repack_sources_kernel(const float4 *__restrict__ pos_mass, int64_t n,
                                                             int64_t n_pad, float4 *__restrict__ packed) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (2 * p >= n_pad) return;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    const float4 b0 = (2 * p < n) ? __ldg(pos_mass + 2 * p) : zero;
    const float4 b1 = (2 * p + 1 < n) ? __ldg(pos_mass + 2 * p + 1) : zero;
    packed[2 * p] = make_float4(b0.x, b1.x, b0.y, b1.y);
    packed[2 * p + 1] = make_float4(b0.z, b1.z, b0.w, b1.w);
}

// ---- the force kernel -----------------------------------------------------------------------------
// Template: I = targets per thread, TJ = sources per shared-memory tile (= accumulation block),
// NST = ring stages, POT = also accumulate sum_j m_j / sqrt(r^2+eps^2), MINB = CTAs per SM.
// grid = (target tiles, source splits); block = THREADS.
//   targets of CTA bx : t0 + bx*THREADS*I + i*THREADS + tid,  i < I   (coalesced loads/stores)
//   sources of split by: packed pairs [by*tiles_per_split*TJ/2, ...), tiles_per_split tiles
// Output: out[(by * out_stride) + target] = (sum_x, sum_y, sum_z, sum_pot) * scale  (scale = G when
// there is a single split and the result is final, else 1 and the reduce kernel applies G).
constexpr int FORCE_THREADS = 256;

template <int I, int TJ, int NST, bool POT, int MINB>
__global__ void __launch_bounds__(FORCE_THREADS, MINB)
force_kernel(const float4 *__restrict__ pos_mass, const float4 *__restrict__ packed, int64_t t_begin,
             int64_t t_count, int tiles_per_split, float eps2, float scale, int final_out,
             float4 *__restrict__ out, int64_t out_stride) {
    constexpr int TILE_BYTES = TJ * 16;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    ulonglong2 *tile = reinterpret_cast<ulonglong2 *>(smem_raw);                    // [NST][TJ] ulonglong2 (= TJ/2 pairs x 2)
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem_raw + NST * TILE_BYTES);  // [NST]
    uint64_t *empty_bar = full_bar + NST;                                            // [NST]

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const unsigned char *src =
        reinterpret_cast<const unsigned char *>(packed) + (size_t)blockIdx.y * tiles_per_split * TILE_BYTES;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], FORCE_THREADS / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s)
            if (s < tiles_per_split) {
                mbar_arrive_expect_tx(&full_bar[s], TILE_BYTES);
                bulk_copy_g2s(smem_raw + s * TILE_BYTES, src + (size_t)s * TILE_BYTES, TILE_BYTES, &full_bar[s]);
            }
    }

    // targets: negated and duplicated so that d = x_j + (-x_k) is one packed add
    u64 nx[I], ny[I], nz[I];
    const int64_t tbase = (int64_t)blockIdx.x * (FORCE_THREADS * I) + tid;
    float self_m[I];
#pragma unroll
    for (int i = 0; i < I; ++i) {
        const int64_t t = tbase + (int64_t)i * FORCE_THREADS;
        float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
        if (t < t_count) b = __ldg(pos_mass + t_begin + t);
        nx[i] = pack2(-b.x, -b.x);
        ny[i] = pack2(-b.y, -b.y);
        nz[i] = pack2(-b.z, -b.z);
        self_m[i] = b.w;
    }
    const u64 eps2_2 = pack2(eps2, eps2);

    float sx[I], sy[I], sz[I], sp[I];   // second-level accumulators (one add per tile)
#pragma unroll
    for (int i = 0; i < I; ++i) sx[i] = sy[i] = sz[i] = sp[i] = 0.f;

    for (int t = 0; t < tiles_per_split; ++t) {
        const int stage = t % NST;
        const uint32_t parity = (t / NST) & 1;
        mbar_wait(&full_bar[stage], parity);
        const ulonglong2 *tp = tile + (size_t)stage * TJ;

        u64 ax[I], ay[I], az[I], ap[I];
#pragma unroll
        for (int i = 0; i < I; ++i) ax[i] = ay[i] = az[i] = ap[i] = 0ull;   // (+0.f, +0.f)

#pragma unroll 4
        for (int p = 0; p < TJ / 2; ++p) {
            const ulonglong2 A = tp[2 * p];       // (x0,x1) (y0,y1)
            const ulonglong2 B = tp[2 * p + 1];   // (z0,z1) (m0,m1)
#pragma unroll
            for (int i = 0; i < I; ++i) {
                const u64 dx = add2(A.x, nx[i]);
                const u64 dy = add2(A.y, ny[i]);
                const u64 dz = add2(B.x, nz[i]);
                u64 r2 = fma2(dx, dx, eps2_2);
                r2 = fma2(dy, dy, r2);
                r2 = fma2(dz, dz, r2);
                float r2a, r2b;
                unpack2(r2, r2a, r2b);
                const u64 rinv = pack2(rsqrt_approx(r2a), rsqrt_approx(r2b));
                const u64 rinv2 = mul2(rinv, rinv);
                const u64 mr = mul2(B.y, rinv);
                const u64 w = mul2(mr, rinv2);
                ax[i] = fma2(w, dx, ax[i]);
                ay[i] = fma2(w, dy, ay[i]);
                az[i] = fma2(w, dz, az[i]);
                if (POT) ap[i] = add2(ap[i], mr);
            }
        }
        // release the stage, refill it with tile t+NST
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[stage]);
        if (tid == 0 && t + NST < tiles_per_split) {
            mbar_wait(&empty_bar[stage], parity);
            mbar_arrive_expect_tx(&full_bar[stage], TILE_BYTES);
            bulk_copy_g2s(smem_raw + stage * TILE_BYTES, src + (size_t)(t + NST) * TILE_BYTES, TILE_BYTES,
                          &full_bar[stage]);
        }
        // flush: even-source + odd-source halves, then into the per-split sum
#pragma unroll
        for (int i = 0; i < I; ++i) {
            float lo, hi;
            unpack2(ax[i], lo, hi);
            sx[i] += lo + hi;
            unpack2(ay[i], lo, hi);
            sy[i] += lo + hi;
            unpack2(az[i], lo, hi);
            sz[i] += lo + hi;
            if (POT) {
                unpack2(ap[i], lo, hi);
                sp[i] += lo + hi;
            }
        }
    }

    float4 *o = out + (size_t)blockIdx.y * out_stride;
#pragma unroll
    for (int i = 0; i < I; ++i) {
        const int64_t t = tbase + (int64_t)i * FORCE_THREADS;
        if (t < t_count) {
            float pot = 0.f;
            if (POT) {
                pot = sp[i];
                // the j = k term m_k / eps was included by the branch-free loop: remove it once, when final
                if (final_out) pot = -(pot - self_m[i] * rsqrt_approx(eps2));
            }
            o[t] = make_float4(sx[i] * scale, sy[i] * scale, sz[i] * scale, pot * scale);
        }
    }
}

// ---- fixed-order reduction of the source-split partials, applies G ---------------------------------
template <bool POT>
__global__ void __launch_bounds__(256) reduce_partials_kernel(const float4 *__restrict__ partial, int64_t stride,
                                                             int splits, int64_t t_count, float G, float eps2,
                                                             const float4 *__restrict__ pos_mass, int64_t t_begin,
                                                             float4 *__restrict__ out) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= t_count) return;
    float4 s = partial[t];
    for (int k = 1; k < splits; ++k) {
        const float4 q = partial[(size_t)k * stride + t];
        s.x += q.x;
        s.y += q.y;
        s.z += q.z;
        s.w += q.w;
    }
    float pot = 0.f;
    if (POT) {
        const float mk = __ldg(pos_mass + t_begin + t).w;
        pot = -(s.w - mk * rsqrt_approx(eps2)) * G;
    }
    out[t] = make_float4(s.x * G, s.y * G, s.z * G, pot);
}

}  // namespace colatus
