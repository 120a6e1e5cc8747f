// force_sym_kernels.cuh -- eq. (1) of arXiv 1208.3444 with every pair evaluated ONCE.
//
//   F_k = G * sum_{j != k} m_j (x_j - x_k) / (|x_j - x_k|^2 + eps^2)^{3/2}
//
// The pair term g_kj = (x_j - x_k) / (r^2 + eps^2)^{3/2} is antisymmetric: body k receives +m_j g_kj and body j
// receives -m_k g_kj (Newton's third law).  The one-directional kernel of force_kernels.cuh evaluates g twice;
// this kernel evaluates it once and applies it to both bodies, for whole-range evaluations (targets = sources):
//
//   * bodies are cut into NB blocks of BT = 512*IP (the targets one CTA keeps in registers, as in force_kernel;
//     IP = 8: 16 targets per thread, 254 registers, one CTA per SM, from 65536 bodies on; IP = 2 below);
//     block a is paired with the H = (NB-1)/2 blocks b = a+1 .. a+H (mod NB) -- a circulant half, so every block
//     has the same amount of work and every unordered block pair is visited exactly once -- plus, one-directionally
//     (plain tile body, reaction ignored), with itself and, when NB is even, with the antipodal block a + NB/2;
//   * inside a symmetric tile the target side accumulates in registers exactly as before; the source side needs
//     the sum over all targets of the CTA.  Per source a lane first adds up its own 2*IP targets, then the warp
//     reduces 8 sources at a time with a TRANSPOSED shuffle tree: at unrolled position p lane l works on source
//     p ^ f(l), f(l) = (l >> 2) & 7, so at every level of the tree the value to keep and the value to send sit in
//     fixed registers (no selects): v[p] += shfl_xor(v[p + h], 4h), h = 4, 2, 1, then two full levels (xor 2, 1).
//     9 shuffles + 9 adds per component per 8 sources; the order is fixed, so results are reproducible bit for bit;
//   * per-warp reaction sums live in shared memory (private to the warp), are added over the 8 warps in fixed
//     order at the end of the tile and written to a row of their own: row S + k - 1 for block distance k.  The
//     fixed-order sum over the S target-side rows and the H reaction rows is the existing partial-sum reduction.
//
// FMA-pipe work per pair: 16 packed ops per (target pair, source) = 4 pair-interactions (14 for equal masses)
// against 24 (22) for two one-directional evaluations.
#pragma once
#include "force_kernels.cuh"

namespace colatus {

template <int IP, int TJ, int NST>
constexpr size_t force_sym_smem_bytes() {
    return (size_t)NST * TJ * 16 + 2 * NST * sizeof(uint64_t) + (size_t)IP * 3 * FORCE_THREADS * 8 +
           (size_t)3 * (FORCE_THREADS / 32) * TJ * 4;
}

// One source tile against the thread's target pairs, both directions.  racc = this warp's reaction sums
// [3][TJ] (x, y, z rows).  mi = the masses of the thread's own target pairs (general loop only).
template <int IP, int TJ, bool EQM>
__device__ __forceinline__ void sym_tile_body(const unsigned char *tile, const u64 (&nx)[IP], const u64 (&ny)[IP],
                                              const u64 (&nz)[IP], const u64 (&mi)[IP], u64 eps2_2, u64 (&ax)[IP],
                                              u64 (&ay)[IP], u64 (&az)[IP], float *racc, int lane) {
    const int f = (lane >> 2) & 7;
    // Position p reads source p ^ f of the 128-byte row of 8 sources.  Two ways to form the address, measured on the
    // B200 (N = 2^20, % of peak by the 20-flop convention): eight per-lane byte offsets (p ^ f) * 16 kept in registers
    // (equal-mass body: 104.4 against 102.8), or the lane's row pointer plus a per-bit signed offset -- p ^ f =
    // f + sum over the set bits b of p of (f has b ? -b : +b) -- which needs no extra registers (general body:
    // 94.2 against 91.5); the first formulation, ((jb + p) ^ f) << 4 computed per load, gave 92.9 / 101.4.  With 16
    // targets per thread (IP = 8) the registers are gone and the row-pointer form wins for equal masses too
    // (265.7 against 267.1 ms).
    int q[8];
    if (EQM && IP <= 3) {
#pragma unroll
        for (int p = 0; p < 8; ++p) q[p] = (p << 4) ^ (f << 4);
    }
    for (int jb = 0; jb < TJ; jb += 8) {
        float vx[8], vy[8], vz[8];
        const unsigned char *row = tile + (jb << 4) + (f << 4);   // this lane's source at position 0
#pragma unroll
        for (int p = 0; p < 8; ++p) {
            const int off = ((p & 1) ? ((f & 1) ? -16 : 16) : 0) + ((p & 2) ? ((f & 2) ? -32 : 32) : 0) +
                            ((p & 4) ? ((f & 4) ? -64 : 64) : 0);
            const float4 S = (EQM && IP <= 3) ? *reinterpret_cast<const float4 *>(tile + (jb << 4) + q[p])
                                              : *reinterpret_cast<const float4 *>(row + off);
            const u64 X = pack2(S.x, S.x), Y = pack2(S.y, S.y), Z = pack2(S.z, S.z), M = pack2(S.w, S.w);
            u64 rx = 0ull, ry = 0ull, rz = 0ull;
#pragma unroll
            for (int i = 0; i < IP; ++i) {
                const u64 dx = add2(nx[i], X);
                const u64 dy = add2(ny[i], Y);
                const u64 dz = add2(nz[i], Z);
                u64 r2 = fma2(dz, dz, eps2_2);
                r2 = fma2(dy, dy, r2);
                r2 = fma2(dx, dx, r2);
                float r2a, r2b;
                unpack2(r2, r2a, r2b);
                const u64 rinv = pack2(rsqrt_approx(r2a), rsqrt_approx(r2b));
                const u64 rinv2 = mul2(rinv, rinv);
                const u64 r3 = mul2(rinv, rinv2);
                const u64 wi = EQM ? r3 : mul2(r3, M);
                const u64 wj = EQM ? r3 : mul2(r3, mi[i]);
                ax[i] = fma2(wi, dx, ax[i]);
                ay[i] = fma2(wi, dy, ay[i]);
                az[i] = fma2(wi, dz, az[i]);
                rx = fma2(wj, dx, rx);
                ry = fma2(wj, dy, ry);
                rz = fma2(wj, dz, rz);
            }
            float lo, hi;
            unpack2(rx, lo, hi);
            vx[p] = lo + hi;
            unpack2(ry, lo, hi);
            vy[p] = lo + hi;
            unpack2(rz, lo, hi);
            vz[p] = lo + hi;
        }
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            vx[p] += __shfl_xor_sync(0xffffffffu, vx[p + 4], 16);
            vy[p] += __shfl_xor_sync(0xffffffffu, vy[p + 4], 16);
            vz[p] += __shfl_xor_sync(0xffffffffu, vz[p + 4], 16);
        }
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            vx[p] += __shfl_xor_sync(0xffffffffu, vx[p + 2], 8);
            vy[p] += __shfl_xor_sync(0xffffffffu, vy[p + 2], 8);
            vz[p] += __shfl_xor_sync(0xffffffffu, vz[p + 2], 8);
        }
        vx[0] += __shfl_xor_sync(0xffffffffu, vx[1], 4);
        vy[0] += __shfl_xor_sync(0xffffffffu, vy[1], 4);
        vz[0] += __shfl_xor_sync(0xffffffffu, vz[1], 4);
        vx[0] += __shfl_xor_sync(0xffffffffu, vx[0], 2);
        vy[0] += __shfl_xor_sync(0xffffffffu, vy[0], 2);
        vz[0] += __shfl_xor_sync(0xffffffffu, vz[0], 2);
        vx[0] += __shfl_xor_sync(0xffffffffu, vx[0], 1);
        vy[0] += __shfl_xor_sync(0xffffffffu, vy[0], 1);
        vz[0] += __shfl_xor_sync(0xffffffffu, vz[0], 1);
        if ((lane & 3) == 0) {                           // lane l now holds the warp's sum for source jb + f(l)
            racc[jb + f] += vx[0];
            racc[TJ + jb + f] += vy[0];
            racc[2 * TJ + jb + f] += vz[0];
        }
    }
}

// Position p of block a's tile list in one launch -> (source tile index, block distance k; k = 0: plain tile).
// A launch covers the block distances k_begin .. k_begin + k_count - 1 and, if `with_plain`, the one-directional
// blocks (the block itself first, the antipodal block last when NB is even).
struct SymTile {
    int tile;   // index of the TJ-source tile in the staged array
    int k;      // 0 = one-directional (diagonal or antipodal block), else symmetric with block distance k
    int sub;    // tile within the block
};
template <int TPB>
__device__ __forceinline__ SymTile sym_tile_at(int p, int a, int nb, int k_begin, int k_count, int with_plain) {
    SymTile t;
    const int lead = with_plain ? TPB : 0;
    int b;
    if (p < lead) {
        t.k = 0;
        t.sub = p;
        b = a;
    } else if (p < lead + TPB * k_count) {
        const int q = p - lead;
        const int dk = q / TPB;
        t.k = k_begin + dk;
        t.sub = q - dk * TPB;
        b = a + t.k;
    } else {
        t.k = 0;
        t.sub = p - lead - TPB * k_count;
        b = a + nb / 2;
    }
    if (b >= nb) b -= nb;
    t.tile = b * TPB + t.sub;
    return t;
}

// grid = (blocks of this launch, S splits): target blocks a_begin .. a_begin + gridDim.x - 1 of the NB blocks (all of
// them for a whole evaluation; a share of them when the evaluation is divided over GPUs or calls,
// colatus_forces_symmetric_part).  staged = the source array padded to NB * BT bodies (far-away zero-mass padding);
// targets are read from it too.  Split s works on positions [s * P / S, (s + 1) * P / S) of the block's list of
// P = TPB * (k_count + (with_plain ? 1 + (NB even) : 0)) tiles.  Output rows of `stride` float4: row s =
// target-side sums of split s (all NB * BT targets); row S + (k - k_begin) = reaction sums (already negated) of
// block distance k.  A launch over all NB blocks writes every row in full; a launch over a share of the blocks writes
// the target-side rows of its own blocks and, in reaction row k, the blocks b = a + k (mod NB) of its blocks a --
// reduce_sym_part_kernel adds exactly those cells.
// BODY: 0 = both tile bodies in the kernel, picked by the equal-mass flag; 1 = general body only, 2 = equal-mass
// body only -- such a kernel returns at once when the flag asks for the other body, so launching the pair (1, 2) is
// the same evaluation with each body scheduled by ptxas on its own (the two bodies in one kernel cost each other
// 1-2.5 %); worth the second, empty launch for large problems only.
// PART: the launch covers the target blocks a_begin .. a_begin + gridDim.x - 1 only (a share of the evaluation).  A
// template parameter, and a_begin the LAST argument, because the mere use of a_begin in the whole-evaluation kernel
// moved ptxas's schedule of the tile loop: 319.3 ms against 313.7 ms at N = 2^20 (round-2 A/B, git history, commit 3dbce46).
template <int IP, int TJ, int NST, int MINB, int BODY, bool PART>
__global__ void __launch_bounds__(FORCE_THREADS, MINB)
force_sym_kernel(const float4 *__restrict__ staged, int nb, int splits, int k_begin, int k_count, int with_plain,
                 float eps2, float4 *__restrict__ partial, int64_t stride, const int *__restrict__ mass_flag,
                 int generation, int *__restrict__ step_ctr, int a_begin) {
    constexpr int TILE_BYTES = TJ * 16;
    constexpr int BT = FORCE_THREADS * 2 * IP;
    constexpr int TPB = BT / TJ;
    constexpr int NW = FORCE_THREADS / 32;
    static_assert(BT % TJ == 0, "a block is a whole number of tiles");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem_raw + NST * TILE_BYTES);
    uint64_t *empty_bar = full_bar + NST;
    u64 *acc2 = reinterpret_cast<u64 *>(smem_raw + NST * TILE_BYTES + 2 * NST * 8);   // [IP*3][THREADS]
    float *racc_all = reinterpret_cast<float *>(acc2 + (size_t)IP * 3 * FORCE_THREADS);   // [NW][3][TJ]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int a = PART ? a_begin + (int)blockIdx.x : (int)blockIdx.x, s = blockIdx.y;
    if (BODY != 0) {                 // uniform over the grid; before any barrier or copy is set up
        griddep_wait();
        if ((__ldcg(mass_flag) != generation) != (BODY == 2)) return;
    }
    const int P = TPB * (k_count + (with_plain ? ((nb & 1) ? 1 : 2) : 0));
    const int p0 = (int)(((int64_t)s * P) / splits), p1 = (int)(((int64_t)(s + 1) * P) / splits);
    const unsigned char *src = reinterpret_cast<const unsigned char *>(staged);

    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < NST; ++q) {
            mbar_init(&full_bar[q], 1);
            mbar_init(&empty_bar[q], NW);
        }
        mbar_fence_init();
    }
    __syncthreads();
    griddep_wait();
    griddep_launch_dependents();
    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < NST; ++q)
            if (p0 + q < p1) {
                const SymTile t = sym_tile_at<TPB>(p0 + q, a, nb, k_begin, k_count, with_plain);
                mbar_arrive_expect_tx(&full_bar[q], TILE_BYTES);
                bulk_copy_g2s(smem_raw + q * TILE_BYTES, src + (size_t)t.tile * TILE_BYTES, TILE_BYTES, &full_bar[q]);
            }
    }

    u64 nx[IP], ny[IP], nz[IP], mi[IP];
    const int64_t tbase = (int64_t)a * BT + 2 * tid;
#pragma unroll
    for (int i = 0; i < IP; ++i) {
        const int64_t t = tbase + (int64_t)i * (2 * FORCE_THREADS);
        const float4 b0 = __ldcg(staged + t), b1 = __ldcg(staged + t + 1);
        nx[i] = pack2(-b0.x, -b1.x);
        ny[i] = pack2(-b0.y, -b1.y);
        nz[i] = pack2(-b0.z, -b1.z);
        mi[i] = pack2(b0.w, b1.w);
    }
    const u64 eps2_2 = pack2(eps2, eps2);
#pragma unroll
    for (int c = 0; c < IP * 3; ++c) acc2[c * FORCE_THREADS + tid] = 0ull;
    float *racc = racc_all + (size_t)warp * 3 * TJ;
    for (int j = lane; j < 3 * TJ; j += 32) racc[j] = 0.f;
    if (step_ctr && tid == FORCE_THREADS - 1 && blockIdx.x == 0 && s == 0) step_ctr[1] = step_ctr[0];
    const bool eqm = __ldcg(mass_flag) != generation;
    const float m_common = eqm ? __ldcg(staged).w : 1.0f;        // applied once to the finished sums
    __syncwarp();

    for (int p = p0; p < p1; ++p) {
        const int it = p - p0;
        const int stage = it % NST;
        const uint32_t parity = (it / NST) & 1;
        const SymTile T = sym_tile_at<TPB>(p, a, nb, k_begin, k_count, with_plain);
        mbar_wait(&full_bar[stage], parity);
        const unsigned char *tile = smem_raw + (size_t)stage * TILE_BYTES;
        u64 ax[IP], ay[IP], az[IP], ap[IP];
#pragma unroll
        for (int i = 0; i < IP; ++i) ax[i] = ay[i] = az[i] = ap[i] = 0ull;
        if (T.k == 0) {
            const float4 *tp = reinterpret_cast<const float4 *>(tile);
            if (BODY == 2 || (BODY == 0 && eqm))
                force_tile_body<IP, TJ, false, true>(tp, nx, ny, nz, eps2_2, ax, ay, az, ap);
            else
                force_tile_body<IP, TJ, false, false>(tp, nx, ny, nz, eps2_2, ax, ay, az, ap);
        } else {
            if (BODY == 2 || (BODY == 0 && eqm))
                sym_tile_body<IP, TJ, true>(tile, nx, ny, nz, mi, eps2_2, ax, ay, az, racc, lane);
            else
                sym_tile_body<IP, TJ, false>(tile, nx, ny, nz, mi, eps2_2, ax, ay, az, racc, lane);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[stage]);
        if (tid == 0 && p + NST < p1) {
            const SymTile N = sym_tile_at<TPB>(p + NST, a, nb, k_begin, k_count, with_plain);
            mbar_wait(&empty_bar[stage], parity);
            mbar_arrive_expect_tx(&full_bar[stage], TILE_BYTES);
            bulk_copy_g2s(smem_raw + stage * TILE_BYTES, src + (size_t)N.tile * TILE_BYTES, TILE_BYTES,
                          &full_bar[stage]);
        }
#pragma unroll
        for (int i = 0; i < IP; ++i) {
            u64 *a2 = acc2 + (size_t)(i * 3) * FORCE_THREADS + tid;
            a2[0] = add2(a2[0], ax[i]);
            a2[FORCE_THREADS] = add2(a2[FORCE_THREADS], ay[i]);
            a2[2 * FORCE_THREADS] = add2(a2[2 * FORCE_THREADS], az[i]);
        }
        if (T.k != 0) {
            // reaction of this tile: add the 8 warps' sums in warp order, negate, write the row of distance k
            __syncthreads();
            int bb = a + T.k;
            if (bb >= nb) bb -= nb;
            float4 *row = partial + (size_t)(splits + T.k - k_begin) * stride + (size_t)bb * BT + (size_t)T.sub * TJ;
            for (int j = tid; j < TJ; j += FORCE_THREADS) {
                float sx = racc_all[j], sy = racc_all[TJ + j], sz = racc_all[2 * TJ + j];
#pragma unroll
                for (int w = 1; w < NW; ++w) {
                    sx += racc_all[(size_t)w * 3 * TJ + j];
                    sy += racc_all[(size_t)w * 3 * TJ + TJ + j];
                    sz += racc_all[(size_t)w * 3 * TJ + 2 * TJ + j];
                }
                row[j] = make_float4(-sx * m_common, -sy * m_common, -sz * m_common, 0.f);
#pragma unroll
                for (int w = 0; w < NW; ++w) {
                    racc_all[(size_t)w * 3 * TJ + j] = 0.f;
                    racc_all[(size_t)w * 3 * TJ + TJ + j] = 0.f;
                    racc_all[(size_t)w * 3 * TJ + 2 * TJ + j] = 0.f;
                }
            }
            __syncthreads();
        }
    }

    float4 *o = partial + (size_t)s * stride;
#pragma unroll
    for (int i = 0; i < IP; ++i) {
        const int64_t t = tbase + (int64_t)i * (2 * FORCE_THREADS);
        const u64 *a2 = acc2 + (size_t)(i * 3) * FORCE_THREADS + tid;
        float fx[2], fy[2], fz[2];
        unpack2(a2[0], fx[0], fx[1]);
        unpack2(a2[FORCE_THREADS], fy[0], fy[1]);
        unpack2(a2[2 * FORCE_THREADS], fz[0], fz[1]);
        o[t] = make_float4(fx[0] * m_common, fy[0] * m_common, fz[0] * m_common, 0.f);
        o[t + 1] = make_float4(fx[1] * m_common, fy[1] * m_common, fz[1] * m_common, 0.f);
    }
}

// ---- the same evaluation with the potential (colatus_forces_potential, the W of colatus_diagnostics) -----------------
template <int IP, int TJ, int NST>
constexpr size_t force_sym_pot_smem_bytes() {
    return (size_t)NST * TJ * 16 + 2 * NST * sizeof(uint64_t) + (size_t)IP * 4 * FORCE_THREADS * 8 +
           (size_t)4 * (FORCE_THREADS / 32) * TJ * 4;
}

// sym_tile_body with the potential as a fourth component: racc = this warp's reaction sums [4][TJ] (x, y, z, pot).
// A function of its own (and a kernel of its own below) rather than a template flag of sym_tile_body: any edit of
// that function's text, even one compiled out, moves ptxas's schedule of the force-only loop (round-2 A/B, git history, commit 3dbce46).  mi = the masses of the thread's own target pairs (general
// loop only).  POT: also sum_j m_j / sqrt(r^2 + eps^2) on the target side and sum_k m_k / sqrt(...) on the source side
// (the potential is symmetric in the pair, not antisymmetric: no sign change for the reaction).
template <int IP, int TJ, bool EQM>
__device__ __forceinline__ void sym_tile_body_pot(const unsigned char *tile, const u64 (&nx)[IP], const u64 (&ny)[IP],
                                              const u64 (&nz)[IP], const u64 (&mi)[IP], u64 eps2_2, u64 (&ax)[IP],
                                              u64 (&ay)[IP], u64 (&az)[IP], u64 (&ap)[IP], float *racc, int lane) {
    const int f = (lane >> 2) & 7;
    // Position p reads source p ^ f of the 128-byte row of 8 sources.  Two ways to form the address, measured on the
    // B200 (N = 2^20, % of peak by the 20-flop convention): eight per-lane byte offsets (p ^ f) * 16 kept in registers
    // (equal-mass body: 104.4 against 102.8), or the lane's row pointer plus a per-bit signed offset -- p ^ f =
    // f + sum over the set bits b of p of (f has b ? -b : +b) -- which needs no extra registers (general body:
    // 94.2 against 91.5); the first formulation, ((jb + p) ^ f) << 4 computed per load, gave 92.9 / 101.4.
    constexpr bool POT = true;
    int q[8];
    if (EQM) {
#pragma unroll
        for (int p = 0; p < 8; ++p) q[p] = (p << 4) ^ (f << 4);
    }
    for (int jb = 0; jb < TJ; jb += 8) {
        float vx[8], vy[8], vz[8], vp[POT ? 8 : 1];
        const unsigned char *row = tile + (jb << 4) + (f << 4);   // this lane's source at position 0
#pragma unroll
        for (int p = 0; p < 8; ++p) {
            const int off = ((p & 1) ? ((f & 1) ? -16 : 16) : 0) + ((p & 2) ? ((f & 2) ? -32 : 32) : 0) +
                            ((p & 4) ? ((f & 4) ? -64 : 64) : 0);
            const float4 S = EQM ? *reinterpret_cast<const float4 *>(tile + (jb << 4) + q[p])
                                 : *reinterpret_cast<const float4 *>(row + off);
            const u64 X = pack2(S.x, S.x), Y = pack2(S.y, S.y), Z = pack2(S.z, S.z), M = pack2(S.w, S.w);
            u64 rx = 0ull, ry = 0ull, rz = 0ull, rp = 0ull;
#pragma unroll
            for (int i = 0; i < IP; ++i) {
                const u64 dx = add2(nx[i], X);
                const u64 dy = add2(ny[i], Y);
                const u64 dz = add2(nz[i], Z);
                u64 r2 = fma2(dz, dz, eps2_2);
                r2 = fma2(dy, dy, r2);
                r2 = fma2(dx, dx, r2);
                float r2a, r2b;
                unpack2(r2, r2a, r2b);
                const u64 rinv = pack2(rsqrt_approx(r2a), rsqrt_approx(r2b));
                const u64 rinv2 = mul2(rinv, rinv);
                const u64 r3 = mul2(rinv, rinv2);
                const u64 wi = EQM ? r3 : mul2(r3, M);
                const u64 wj = EQM ? r3 : mul2(r3, mi[i]);
                ax[i] = fma2(wi, dx, ax[i]);
                ay[i] = fma2(wi, dy, ay[i]);
                az[i] = fma2(wi, dz, az[i]);
                rx = fma2(wj, dx, rx);
                ry = fma2(wj, dy, ry);
                rz = fma2(wj, dz, rz);
                if (POT) {
                    ap[i] = add2(ap[i], EQM ? rinv : mul2(rinv, M));
                    rp = EQM ? add2(rp, rinv) : fma2(rinv, mi[i], rp);
                }
            }
            float lo, hi;
            unpack2(rx, lo, hi);
            vx[p] = lo + hi;
            unpack2(ry, lo, hi);
            vy[p] = lo + hi;
            unpack2(rz, lo, hi);
            vz[p] = lo + hi;
            if (POT) {
                unpack2(rp, lo, hi);
                vp[p] = lo + hi;
            }
        }
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            vx[p] += __shfl_xor_sync(0xffffffffu, vx[p + 4], 16);
            vy[p] += __shfl_xor_sync(0xffffffffu, vy[p + 4], 16);
            vz[p] += __shfl_xor_sync(0xffffffffu, vz[p + 4], 16);
            if (POT) vp[p] += __shfl_xor_sync(0xffffffffu, vp[POT ? p + 4 : 0], 16);
        }
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            vx[p] += __shfl_xor_sync(0xffffffffu, vx[p + 2], 8);
            vy[p] += __shfl_xor_sync(0xffffffffu, vy[p + 2], 8);
            vz[p] += __shfl_xor_sync(0xffffffffu, vz[p + 2], 8);
            if (POT) vp[p] += __shfl_xor_sync(0xffffffffu, vp[POT ? p + 2 : 0], 8);
        }
        vx[0] += __shfl_xor_sync(0xffffffffu, vx[1], 4);
        vy[0] += __shfl_xor_sync(0xffffffffu, vy[1], 4);
        vz[0] += __shfl_xor_sync(0xffffffffu, vz[1], 4);
        vx[0] += __shfl_xor_sync(0xffffffffu, vx[0], 2);
        vy[0] += __shfl_xor_sync(0xffffffffu, vy[0], 2);
        vz[0] += __shfl_xor_sync(0xffffffffu, vz[0], 2);
        vx[0] += __shfl_xor_sync(0xffffffffu, vx[0], 1);
        vy[0] += __shfl_xor_sync(0xffffffffu, vy[0], 1);
        vz[0] += __shfl_xor_sync(0xffffffffu, vz[0], 1);
        if (POT) {
            vp[0] += __shfl_xor_sync(0xffffffffu, vp[POT ? 1 : 0], 4);
            vp[0] += __shfl_xor_sync(0xffffffffu, vp[0], 2);
            vp[0] += __shfl_xor_sync(0xffffffffu, vp[0], 1);
        }
        if ((lane & 3) == 0) {                           // lane l now holds the warp's sum for source jb + f(l)
            racc[jb + f] += vx[0];
            racc[TJ + jb + f] += vy[0];
            racc[2 * TJ + jb + f] += vz[0];
            if (POT) racc[3 * TJ + jb + f] += vp[0];
        }
    }
}

// POT: rows carry the potential sums in .w (target side: sum_j m_j / sqrt(r^2 + eps^2) including the j = k term of the
// diagonal tiles, which the row reduction removes; reaction rows: the same sum over the block's partners).
template <int IP, int TJ, int NST, int MINB>
__global__ void __launch_bounds__(FORCE_THREADS, MINB)
force_sym_pot_kernel(const float4 *__restrict__ staged, int nb, int splits, int k_begin, int k_count, int with_plain,
                 float eps2, float4 *__restrict__ partial, int64_t stride, const int *__restrict__ mass_flag,
                 int generation) {
    constexpr bool POT = true, PART = false;
    constexpr int BODY = 0;
    int *const step_ctr = nullptr;
    const int a_begin = 0;
    constexpr int TILE_BYTES = TJ * 16;
    constexpr int BT = FORCE_THREADS * 2 * IP;
    constexpr int TPB = BT / TJ;
    constexpr int NW = FORCE_THREADS / 32;
    static_assert(BT % TJ == 0, "a block is a whole number of tiles");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem_raw + NST * TILE_BYTES);
    uint64_t *empty_bar = full_bar + NST;
    constexpr int NC = POT ? 4 : 3;                                                   // components per body
    u64 *acc2 = reinterpret_cast<u64 *>(smem_raw + NST * TILE_BYTES + 2 * NST * 8);   // [IP*NC][THREADS]
    float *racc_all = reinterpret_cast<float *>(acc2 + (size_t)IP * NC * FORCE_THREADS);   // [NW][NC][TJ]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int a = PART ? a_begin + (int)blockIdx.x : (int)blockIdx.x, s = blockIdx.y;
    if (BODY != 0) {                 // uniform over the grid; before any barrier or copy is set up
        griddep_wait();
        if ((__ldcg(mass_flag) != generation) != (BODY == 2)) return;
    }
    const int P = TPB * (k_count + (with_plain ? ((nb & 1) ? 1 : 2) : 0));
    const int p0 = (int)(((int64_t)s * P) / splits), p1 = (int)(((int64_t)(s + 1) * P) / splits);
    const unsigned char *src = reinterpret_cast<const unsigned char *>(staged);

    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < NST; ++q) {
            mbar_init(&full_bar[q], 1);
            mbar_init(&empty_bar[q], NW);
        }
        mbar_fence_init();
    }
    __syncthreads();
    griddep_wait();
    griddep_launch_dependents();
    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < NST; ++q)
            if (p0 + q < p1) {
                const SymTile t = sym_tile_at<TPB>(p0 + q, a, nb, k_begin, k_count, with_plain);
                mbar_arrive_expect_tx(&full_bar[q], TILE_BYTES);
                bulk_copy_g2s(smem_raw + q * TILE_BYTES, src + (size_t)t.tile * TILE_BYTES, TILE_BYTES, &full_bar[q]);
            }
    }

    u64 nx[IP], ny[IP], nz[IP], mi[IP];
    const int64_t tbase = (int64_t)a * BT + 2 * tid;
#pragma unroll
    for (int i = 0; i < IP; ++i) {
        const int64_t t = tbase + (int64_t)i * (2 * FORCE_THREADS);
        const float4 b0 = __ldcg(staged + t), b1 = __ldcg(staged + t + 1);
        nx[i] = pack2(-b0.x, -b1.x);
        ny[i] = pack2(-b0.y, -b1.y);
        nz[i] = pack2(-b0.z, -b1.z);
        mi[i] = pack2(b0.w, b1.w);
    }
    const u64 eps2_2 = pack2(eps2, eps2);
#pragma unroll
    for (int c = 0; c < IP * NC; ++c) acc2[c * FORCE_THREADS + tid] = 0ull;
    float *racc = racc_all + (size_t)warp * NC * TJ;
    for (int j = lane; j < NC * TJ; j += 32) racc[j] = 0.f;
    if (step_ctr && tid == FORCE_THREADS - 1 && blockIdx.x == 0 && s == 0) step_ctr[1] = step_ctr[0];
    const bool eqm = __ldcg(mass_flag) != generation;
    const float m_common = eqm ? __ldcg(staged).w : 1.0f;        // applied once to the finished sums
    __syncwarp();

    for (int p = p0; p < p1; ++p) {
        const int it = p - p0;
        const int stage = it % NST;
        const uint32_t parity = (it / NST) & 1;
        const SymTile T = sym_tile_at<TPB>(p, a, nb, k_begin, k_count, with_plain);
        mbar_wait(&full_bar[stage], parity);
        const unsigned char *tile = smem_raw + (size_t)stage * TILE_BYTES;
        u64 ax[IP], ay[IP], az[IP], ap[IP];
#pragma unroll
        for (int i = 0; i < IP; ++i) ax[i] = ay[i] = az[i] = ap[i] = 0ull;
        if (T.k == 0) {
            const float4 *tp = reinterpret_cast<const float4 *>(tile);
            if (BODY == 2 || (BODY == 0 && eqm))
                force_tile_body<IP, TJ, POT, true>(tp, nx, ny, nz, eps2_2, ax, ay, az, ap);
            else
                force_tile_body<IP, TJ, POT, false>(tp, nx, ny, nz, eps2_2, ax, ay, az, ap);
        } else {
            if (BODY == 2 || (BODY == 0 && eqm))
                sym_tile_body_pot<IP, TJ, true>(tile, nx, ny, nz, mi, eps2_2, ax, ay, az, ap, racc, lane);
            else
                sym_tile_body_pot<IP, TJ, false>(tile, nx, ny, nz, mi, eps2_2, ax, ay, az, ap, racc, lane);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[stage]);
        if (tid == 0 && p + NST < p1) {
            const SymTile N = sym_tile_at<TPB>(p + NST, a, nb, k_begin, k_count, with_plain);
            mbar_wait(&empty_bar[stage], parity);
            mbar_arrive_expect_tx(&full_bar[stage], TILE_BYTES);
            bulk_copy_g2s(smem_raw + stage * TILE_BYTES, src + (size_t)N.tile * TILE_BYTES, TILE_BYTES,
                          &full_bar[stage]);
        }
#pragma unroll
        for (int i = 0; i < IP; ++i) {
            u64 *a2 = acc2 + (size_t)(i * NC) * FORCE_THREADS + tid;
            a2[0] = add2(a2[0], ax[i]);
            a2[FORCE_THREADS] = add2(a2[FORCE_THREADS], ay[i]);
            a2[2 * FORCE_THREADS] = add2(a2[2 * FORCE_THREADS], az[i]);
            if (POT) a2[3 * FORCE_THREADS] = add2(a2[3 * FORCE_THREADS], ap[i]);
        }
        if (T.k != 0) {
            // reaction of this tile: add the 8 warps' sums in warp order, negate, write the row of distance k
            __syncthreads();
            int bb = a + T.k;
            if (bb >= nb) bb -= nb;
            float4 *row = partial + (size_t)(splits + T.k - k_begin) * stride + (size_t)bb * BT + (size_t)T.sub * TJ;
            for (int j = tid; j < TJ; j += FORCE_THREADS) {
                float sx = racc_all[j], sy = racc_all[TJ + j], sz = racc_all[2 * TJ + j];
                float sp = POT ? racc_all[3 * TJ + j] : 0.f;
#pragma unroll
                for (int w = 1; w < NW; ++w) {
                    sx += racc_all[(size_t)w * NC * TJ + j];
                    sy += racc_all[(size_t)w * NC * TJ + TJ + j];
                    sz += racc_all[(size_t)w * NC * TJ + 2 * TJ + j];
                    if (POT) sp += racc_all[(size_t)w * NC * TJ + 3 * TJ + j];
                }
                row[j] = make_float4(-sx * m_common, -sy * m_common, -sz * m_common, sp * m_common);
#pragma unroll
                for (int w = 0; w < NW; ++w) {
                    racc_all[(size_t)w * NC * TJ + j] = 0.f;
                    racc_all[(size_t)w * NC * TJ + TJ + j] = 0.f;
                    racc_all[(size_t)w * NC * TJ + 2 * TJ + j] = 0.f;
                    if (POT) racc_all[(size_t)w * NC * TJ + 3 * TJ + j] = 0.f;
                }
            }
            __syncthreads();
        }
    }

    float4 *o = partial + (size_t)s * stride;
#pragma unroll
    for (int i = 0; i < IP; ++i) {
        const int64_t t = tbase + (int64_t)i * (2 * FORCE_THREADS);
        const u64 *a2 = acc2 + (size_t)(i * NC) * FORCE_THREADS + tid;
        float fx[2], fy[2], fz[2], fp[2] = {0.f, 0.f};
        unpack2(a2[0], fx[0], fx[1]);
        unpack2(a2[FORCE_THREADS], fy[0], fy[1]);
        unpack2(a2[2 * FORCE_THREADS], fz[0], fz[1]);
        if (POT) unpack2(a2[3 * FORCE_THREADS], fp[0], fp[1]);
        o[t] = make_float4(fx[0] * m_common, fy[0] * m_common, fz[0] * m_common, fp[0] * m_common);
        o[t + 1] = make_float4(fx[1] * m_common, fy[1] * m_common, fz[1] * m_common, fp[1] * m_common);
    }
}

// Later chunks of a chunked POTENTIAL evaluation: out += G * (row sums), with out.w -= G * (potential row sums) -- the
// first chunk went through reduce_partials_kernel<true>, which also removed the j = k term.
__global__ void __launch_bounds__(256)
reduce_sym_pot_more_kernel(const float4 *__restrict__ partial, int64_t stride, int rows, int64_t n, float G,
                           float4 *__restrict__ out) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const float4 s = sum_partials(partial, stride, rows, t);
    float4 o = out[t];
    o.x += s.x * G;
    o.y += s.y * G;
    o.z += s.z * G;
    o.w -= s.w * G;
    out[t] = o;
}

// Fixed-order sum of the cells a launch over target blocks [a_begin, a_begin + a_count) has written (above), for
// every body t < n: the S target-side rows if t's block is one of the launch's, then reaction row k for every block
// distance k of the launch whose source block b - k (mod NB) is one of the launch's.  FP64 accumulation, one rounding,
// x G.  ACCUM adds to out (later chunks of block distances).  Summed over a partition of the blocks, the outputs are
// the whole force: this is what a GPU contributes before the all-reduce of the sharded symmetric evaluation.
template <bool ACCUM>
__global__ void __launch_bounds__(256)
reduce_sym_part_kernel(const float4 *__restrict__ partial, int64_t stride, int splits, int k_begin, int k_count, int nb,
                       int block_bodies, int a_begin, int a_count, int with_plain, int64_t n, float G,
                       float4 *__restrict__ out) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const int b = (int)(t / block_bodies);
    double sx = 0.0, sy = 0.0, sz = 0.0;
    int rel = b - a_begin;
    if (rel < 0) rel += nb;
    if (rel < a_count) {
        (void)with_plain;               // the target-side rows hold 0 for a launch without one-directional tiles too
        for (int s = 0; s < splits; ++s) {
            const float4 q = partial[(size_t)s * stride + t];
            sx += (double)q.x;
            sy += (double)q.y;
            sz += (double)q.z;
        }
    }
    for (int dk = 0; dk < k_count; ++dk) {
        int a = b - (k_begin + dk);
        if (a < 0) a += nb;
        int ra = a - a_begin;
        if (ra < 0) ra += nb;
        if (ra < a_count) {
            const float4 q = partial[(size_t)(splits + dk) * stride + t];
            sx += (double)q.x;
            sy += (double)q.y;
            sz += (double)q.z;
        }
    }
    float4 r = make_float4((float)sx * G, (float)sy * G, (float)sz * G, 0.f);
    if (ACCUM) {
        const float4 o = out[t];
        r.x += o.x;
        r.y += o.y;
        r.z += o.z;
    }
    out[t] = r;
}

}  // namespace colatus
