// colatus_api.cu -- the C-ABI boundary of libcolatus (include/colatus.h): argument validation,
// launch geometry and kernel launches.  All arithmetic of the path lives in the kernels of
// force_kernels.cuh / integrate_kernels.cuh; the host forms only the per-step coefficients.
// Links the CUDA runtime only (no libtorch).  There is no CPU fallback.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <limits>
#include <vector>

#include "../../include/colatus.h"
#include "force_kernels.cuh"
#include "force_sym_kernels.cuh"
#include "integrate_kernels.cuh"
#include "analysis_kernels.cuh"

namespace {

using namespace colatus;

constexpr int MAX_SPLITS = REDUCE_MAX_SPLITS;   // source splits (partials kept in the workspace): small problems
constexpr int MAX_SPLITS_LARGE = 16;            // ... and problems above SMALL_N bodies (bounds the partials' memory)
constexpr int64_t SMALL_N = 65536;
constexpr int NSTAGES = 4;            // shared-memory ring depth
constexpr int DIAG_BLOCKS_MAX = 1024;
constexpr int64_t PAD_SOURCES = 1024; // n_pad granularity = largest tile
constexpr int RUN_CHUNK = 1024;       // steps per coefficient-table upload in colatus_run
#ifndef COLATUS_GRAPH_STEPS
#define COLATUS_GRAPH_STEPS 8
#endif
#ifndef COLATUS_TAIL_THREADS
#define COLATUS_TAIL_THREADS 256
#endif
constexpr int GRAPH_STEPS = COLATUS_GRAPH_STEPS;        // steps per replay of the multi-step graph (two-kernel loop; divides RUN_CHUNK)

// symmetric (each pair once) force kernel, force_sym_kernels.cuh: whole-range evaluations of at least SYM_MIN_N bodies
// Variants: blocks of 4096 bodies (16 targets per thread, 254 registers, ONE CTA per SM, 512-source tiles) from
// SYM_MID_N bodies on -- the per-source work of the source side (shuffle tree, permuted load, address arithmetic) is
// amortised over 16 targets instead of 6 and 8 independent chains per thread replace the second CTA: 292.8 ms against
// 313.8 ms at N = 2^20 (round-2 measurement); below SYM_MID_N blocks of 1024 (4 targets per
// thread, two CTAs per SM, 256-source tiles), whose finer tiles split better over the SMs (section 4b).  The first
// variant written, blocks of 1536 (6 targets per thread, two CTAs per SM), is between the two everywhere (within
// 1 % of the better one at 49152 and 98304 bodies only) and stays selectable ("symmetric_block") for comparisons.
constexpr int64_t SYM_MID_N = 65536;
constexpr int64_t SYM_WIDE_N = SYM_MID_N;
constexpr int64_t SYM_MIN_N = 20480;   // measured: faster than force_kernel from here on (profiles/r02_symmetric_kernel.md)
constexpr int SYM_MAX_SPLITS = 32;
constexpr int64_t SYM_PAIR_N = 98304;                            // from here on: one kernel per tile body (launch_force_sym)
constexpr int SYM_MIN_ROWS = 32;                                  // reaction rows a launch of the 1024 / 1536-body variants can always hold
// Row budget of the wide (4096-body) variant: all rows of an evaluation while they fit 512 MiB, else 32 rows (splits +
// block distances per launch), the evaluation then being chunked over block distances.  Measured knee
// (profiles/r03_workspace_rows_sweep.md): N = 2^20 takes 293.3 ms with all 142 rows (2.4 GB) and 295.3 ms (+0.7 %) with
// 32 rows (0.5 GB, 8 launches); N = 2^22 4673 ms with 128 rows (8 GiB) and 4690 ms (+0.4 %) with 32 (2 GiB, 27 launches).
constexpr size_t SYM_ROWS_BUDGET = (size_t)512 << 20;
constexpr int SYM_BUDGET_ROWS = 32;

struct Geometry {
    int IP = 0, TJ = 0;   // target pairs per thread, sources per tile
    int64_t tiles_t = 0;
    int splits = 0, tiles_per_split = 0;
    int64_t n_pad = 0;   // sources covered = splits * tiles_per_split * TJ
    // symmetric kernel: nb blocks of bt() bodies (n_pad = nb * bt(), tiles_t = nb), H block distances,
    // K of them per launch (K reaction rows + `splits` target-side rows in the workspace), `chunks` launches
    bool sym = false;
    int nb = 0, H = 0, K = 0, chunks = 0;
    int a_begin = 0, a_count = 0;   // target blocks of this evaluation (all nb of them unless it is a share: ..._part)
    int64_t bt() const { return (int64_t)FORCE_THREADS * 2 * IP; }   // bodies per block = targets of one CTA
    int tpb() const { return (int)(bt() / TJ); }                      // tiles per block
};

struct Workspace {     // byte offsets inside the caller's workspace
    size_t packed = 0, partials = 0, scratch_acc = 0, acc64 = 0, trace_slot = 0, diag = 0, stage_in = 0, stage_out = 0,
           step_table = 0, step_ctr = 0, total = 0;
    static constexpr size_t mass_flag = 0;   // first 256 bytes of the workspace: fixed place for every n
};

struct Context {
    bool initialised = false;
    double G = 0.0;
    int device = 0, sm_count = 0, ctas_per_sm = 2;
    unsigned char *ws = nullptr;
    size_t ws_bytes = 0;
    // resident state
    bool uploaded = false;
    float4 *pos = nullptr, *vel = nullptr, *acc = nullptr;
    int64_t n = 0, t_begin = 0, t_count = 0;
    float eps2 = 0.f;
    cudaStream_t stream = nullptr;
    int64_t step = 0;
    // tracers
    int trace_k = 0, trace_cap = 0;
    float4 *ring = nullptr;
    int64_t trace_n = 0;   // n for which the slot map was built
    // instrumentation
    bool profile = false;
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    int64_t launches = 0;
    // tuning overrides (0 = automatic)
    int force_I = 0, force_splits = 0;
    int sym_block = 0;    // 0 = automatic, else 1024, 1536 or 4096 bodies per block ("symmetric_block")
    int sym_rows = 0;     // cap on partial rows per launch of the symmetric kernel (0 = what the workspace holds)
    int symmetric = 1;    // 0 = never, 1 = automatic (n >= SYM_MIN_N), 2 = whenever the evaluation allows it
    int init_epoch = 0;   // counts colatus_init calls
    int generation = 0;   // equal-mass detection stamp (never 0: the flag word starts at 0)
    // external terms: eq. (10) source and mean-density background (0 = off)
    double def_S = 0.0, def_x[3] = {0, 0, 0}, bg_rho = 0.0, bg_c[3] = {0, 0, 0};
    // colatus_run: private capture stream, ordering events, cached one-step graph
    cudaStream_t run_stream = nullptr;
    cudaEvent_t run_ev_in = nullptr, run_ev_out = nullptr;
    cudaGraph_t graph = nullptr, graph_k = nullptr;           // one step / GRAPH_STEPS steps
    cudaGraphExec_t graph_exec = nullptr, graph_exec_k = nullptr;
    bool graph_valid = false;
    int64_t graph_launches = 0;
    int graph_generation = 0;   // equal-mass stamp baked into the captured kernels
    char err[512] = "";
};

Context g;

int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g.err, sizeof(g.err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                              \
    do {                                                                                            \
        cudaError_t e_ = (expr);                                                                    \
        if (e_ != cudaSuccess)                                                                      \
            return fail(COLATUS_CUDA_ERROR, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), \
                        __FILE__, __LINE__);                                                        \
    } while (0)

// Kernel launch with the programmatic-stream-serialization attribute (pdl): the kernel may be scheduled before its
// predecessor in the stream has drained and synchronises with griddepcontrol.wait (force_kernels.cuh).
template <typename... KArgs, typename... Args>
cudaError_t launch_ex(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl,
                      Args &&...args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline int max_splits(int64_t n) { return n <= SMALL_N ? MAX_SPLITS : MAX_SPLITS_LARGE; }

// Bytes of partial-sum rows for n bodies: the source-split partials of force_kernel, and for n >= SYM_MIN_N the
// rows of force_sym_kernel -- all of them ((splits + H) rows of n_pad bodies) while that stays within the budget,
// else the budget (the evaluation is then chunked over block distances).  Non-decreasing in n, so a workspace
// sized for n_max serves every n <= n_max.
inline int sym_ip(int64_t n) { return g.sym_block ? g.sym_block / 512 : (n < SYM_MID_N ? 2 : (n < SYM_WIDE_N ? 3 : 8)); }
inline int64_t sym_blocks(int64_t n, int ip) { return (n + 512 * ip - 1) / (512 * ip); }
size_t sym_rows_bytes(int64_t n, int ip) {
    const size_t row = (size_t)sym_blocks(n, ip) * 512 * ip * 16;
    size_t bytes = ((ip > 3 ? 24 : SYM_MAX_SPLITS) + 2) * row;      // tiny n with "symmetric" = 2: every split count
    if (n >= SYM_MIN_N) {
        const size_t H = (size_t)((sym_blocks(n, ip) - 1) / 2);
        size_t want;
        if (ip > 3) {               // wide variant (n >= SYM_WIDE_N): up to 24 splits; budget as above
            want = (24 + H) * row;
            const size_t budget = SYM_ROWS_BUDGET > SYM_BUDGET_ROWS * row ? SYM_ROWS_BUDGET : SYM_BUDGET_ROWS * row;
            if (want > budget) want = budget;
        } else {                    // automatic below SYM_WIDE_N only (rows of at most 1 MiB): 64 rows hold every plan
            want = (SYM_MAX_SPLITS + H) * row;
            const size_t least = (size_t)(SYM_MAX_SPLITS + SYM_MIN_ROWS) * row;
            if (want < least) want = least;
        }
        if (want > bytes) bytes = want;
    }
    return bytes;
}
// Every variant's need at min(n, the end of the range in which it is the automatic choice) -- forced beyond its
// range ("symmetric_block") a variant gets by with what is there: more launches.  Non-decreasing across the thresholds.
size_t partials_bytes(int64_t n) {
    size_t bytes = (size_t)max_splits(n) * (size_t)n * 16;
    const int64_t n2 = n < SYM_MID_N ? n : SYM_MID_N - 1, n3 = n < SYM_WIDE_N ? n : SYM_WIDE_N - 1;
    if (sym_rows_bytes(n2, 2) > bytes) bytes = sym_rows_bytes(n2, 2);
    if (sym_rows_bytes(n3, 3) > bytes) bytes = sym_rows_bytes(n3, 3);
    if (sym_rows_bytes(n, 8) > bytes) bytes = sym_rows_bytes(n, 8);
    return bytes;
}

Workspace workspace_layout(int64_t n_max) {
    Workspace w;
    const size_t n = (size_t)n_max;
    const size_t n_pad = round_up(n, (size_t)PAD_SOURCES) + (size_t)MAX_SPLITS * PAD_SOURCES;
    size_t off = 256;                        // [0, 256): mass_flag (zeroed by colatus_init)
    w.packed = off;      off += round_up(n_pad * 16, 256);
    w.partials = off;    off += round_up(partials_bytes(n_max), 256);
    w.scratch_acc = off; off += round_up(n * 16, 256);
    w.acc64 = off;       off += round_up(n * 24, 256);      // FP64 running sums of chunked symmetric evaluations
    w.trace_slot = off;  off += round_up(n * 4, 256);
    w.diag = off;        off += round_up((size_t)(DIAG_BLOCKS_MAX + 2) * DIAG_Q * 8, 256);
    w.stage_in = off;    off += round_up(n * 16, 256);
    w.stage_out = off;   off += round_up(n * 16, 256);
    w.step_table = off;  off += round_up((size_t)RUN_CHUNK * sizeof(StepCoef), 256);
    w.step_ctr = off;    off += 256;
    w.total = off;
    return w;
}

// Pick the kernel variant (target pairs per thread, tile) and the source split by a cost model fitted to
// a sweep of every (variant, split) at N = 4096 ... 262144 on the B200 (DESIGN.md 6.3 "Launch geometry";
// round-2 sweep through colatus_set_option, git history, commit 3dbce46: profiles/r02_geometry_sweep.md -- picks within 0.6 % of the best
// measured geometry with <= 16 splits at every size but N = 8192 (+5 %)):
//   time ~ a_IP * IP * S * (per_sm + 0.1) + per_sm * c0
// S = padded sources per split, per_sm = ceil(CTAs / SMs) (an SM works through its CTAs two at a time,
// work-conserving, so what counts is CTAs per SM, not waves of resident slots), a_IP = time per source and
// target pair of a CTA with the SM to itself, c0 = per-CTA prologue/epilogue.  Pure function of
// (n, t_count, SM count): the geometry, and with it the summation order, is reproducible.
Geometry choose_plain_geometry(int64_t n, int64_t t_count) {
    static const int variants[3][2] = {{3, 512}, {2, 512}, {1, 128}};   // (target pairs per thread, tile)
    // per source, per target pair.  a_us[2] was 0.0287 in round 1; the round-2 sweep (same history)
    // shows the 4-targets-per-thread variant level with the 6-target one for equal masses, and 0.0283 moves
    // N = 131072 from 86 x 12 (+3.4 % over the best measured) to 128 x 16 (+0.2 %) with no other pick changed
    static const double a_us[4] = {0.0, 0.0295, 0.0283, 0.0274};
    const double c0_us = 0.77, ramp = 0.096;
    Geometry best;
    double best_cost = -1.0;
    for (int v = 0; v < 3; ++v) {
        const int IP = variants[v][0], TJ = variants[v][1];
        if (g.force_I && g.force_I != 2 * IP) continue;
        const int64_t per_cta = (int64_t)FORCE_THREADS * 2 * IP;
        const int64_t tiles_t = (t_count + per_cta - 1) / per_cta;
        const int64_t src_tiles = (n + TJ - 1) / TJ;
        // automatic choice: at most 16 splits -- the round-2 sweep shows that beyond 16 the
        // growing partial-sum reduction eats what the force kernel gains (<= 1.8 % at best, -35 % at worst);
        // a forced split count (colatus_set_option) may go up to max_splits(n)
        const int64_t cap = g.force_splits ? max_splits(n) : MAX_SPLITS_LARGE;
        const int64_t smax = src_tiles < cap ? src_tiles : cap;
        for (int64_t s = 1; s <= smax; ++s) {
            if (g.force_splits && s != g.force_splits && g.force_splits <= smax) continue;
            const int64_t tps = (src_tiles + s - 1) / s;
            const int64_t units = tiles_t * s;
            const int64_t per_sm = (units + g.sm_count - 1) / g.sm_count;
            const double cost = a_us[IP] * IP * (double)(tps * TJ) * ((double)per_sm + ramp) + (double)per_sm * c0_us;
            if (best_cost < 0.0 || cost < best_cost * 0.998) {   // prefer earlier (fewer splits, more targets) on near ties
                best_cost = cost;
                best.IP = IP;
                best.TJ = TJ;
                best.tiles_t = tiles_t;
                best.splits = (int)s;
                best.tiles_per_split = (int)tps;
                best.n_pad = s * tps * TJ;
            }
        }
    }
    return best;
}

// Symmetric kernel (force_sym_kernels.cuh): whole-range evaluations without the potential, n >= SYM_MIN_N (or
// forced by the "symmetric" option), automatic kernel variant.  nb blocks x S splits CTAs; S from the same kind
// of cost model as above in units of one symmetric tile: (tiles per CTA) * (CTAs per SM + ramp) + CTAs per SM * c0.
// K = block distances per launch = what the partial rows of workspace_layout(n) hold; a pure function of n.
bool sym_eligible(int64_t n, int64_t t_count, bool potential) {
    (void)potential;            // potential evaluations take the symmetric kernel too (its 1024-body variant)
    if (g.symmetric == 0 || t_count != n || g.force_I != 0) return false;
    return g.symmetric == 2 || n >= SYM_MIN_N;
}

Geometry choose_sym_geometry(int64_t n, int part = 0, int parts = 1, bool potential = false) {
    Geometry geo;
    geo.sym = true;
    geo.IP = potential ? 2 : sym_ip(n);      // the potential's fourth component fits the 128 registers with 4 targets/thread
    geo.TJ = geo.IP == 3 ? 512 : 256;
    geo.nb = (int)sym_blocks(n, geo.IP);
    geo.a_begin = (int)((int64_t)geo.nb * part / parts);
    geo.a_count = (int)((int64_t)geo.nb * (part + 1) / parts) - geo.a_begin;
    geo.tiles_t = geo.nb;
    geo.n_pad = (int64_t)geo.nb * geo.bt();
    geo.H = (geo.nb - 1) / 2;
    int64_t rows_avail = (int64_t)(partials_bytes(n) / ((size_t)geo.n_pad * 16));
    if (g.sym_rows >= 2 && g.sym_rows < rows_avail) rows_avail = g.sym_rows;   // "symmetric_rows": forces chunking
    if (rows_avail < 2) {        // (forced on a tiny problem) no room for one target-side and one reaction row
        geo.sym = false;
        return geo;
    }
    const int tpb = geo.tpb();
    const double plain_tiles = tpb * ((geo.nb & 1) ? 1.0 : 2.0) * 0.68;   // a one-directional tile costs ~0.68 symmetric ones
    const double c0 = geo.IP == 2 ? 0.05 : 0.04;                           // per-CTA overhead in units of one tile
    double best_cost = -1.0;
    // more splits than the 16 of the first variant help where the wave count is coarse (one CTA per SM: up to 24) and
    // where a block has few tiles (1024-body blocks: up to 32; N = 32768: kernel 0.335 ms with 32 against 0.363 with 14)
    const int smax = geo.IP > 3 ? 24 : (geo.IP == 2 ? SYM_MAX_SPLITS : 16);
    for (int s = 1; s <= smax; ++s) {
        if (g.force_splits && g.force_splits <= smax && g.force_splits < rows_avail && s != g.force_splits)
            continue;
        if (s >= rows_avail) break;
        int K = (int)(rows_avail - s);
        if (K > geo.H) K = geo.H;
        if (K < 1) K = 1;
        const int chunks = geo.H == 0 ? 1 : (geo.H + K - 1) / K;
        const int64_t ctas = (int64_t)(geo.a_count > 0 ? geo.a_count : 1) * s;
        const double per_sm = (double)((ctas + g.sm_count - 1) / g.sm_count);
        const double tiles = (plain_tiles + (double)tpb * geo.H) / s;
        const double cost = tiles * (per_sm + 0.096) + chunks * per_sm * c0;
        if (best_cost < 0.0 || cost < best_cost * 0.998) {
            best_cost = cost;
            geo.splits = s;
            geo.K = K;
            geo.chunks = chunks;
        }
    }
    geo.tiles_per_split = (int)((tpb * (geo.H + 2) + geo.splits - 1) / geo.splits);
    return geo;
}

Geometry choose_geometry(int64_t n, int64_t t_count, bool potential = false) {
    if (sym_eligible(n, t_count, potential)) {
        const Geometry geo = choose_sym_geometry(n, 0, 1, potential);
        if (geo.sym) return geo;
    }
    return choose_plain_geometry(n, t_count);
}

// One evaluation chunk = one launch of the kernel that holds both tile bodies (general, equal-mass; picked on the
// device), or -- from SYM_PAIR_N bodies on -- two launches, a general-only and an equal-mass-only kernel, of which the
// one the equal-mass flag does not ask for returns at once (15 us at 2^20): compiled alone the general body runs
// 2.4 % faster (94.0 % against 91.8 % of peak at 2^20; the equal-mass body is the same either way).
template <int IP, int TJ, int BODY, bool PART>
cudaError_t launch_force_sym_inst(const Geometry &geo, const float4 *packed, int k_begin, int k_count, int with_plain,
                                  float eps2, float4 *partials, const int *mass_flag, int generation, int *step_ctr,
                                  cudaStream_t st, bool pdl) {
    auto kern = force_sym_kernel<IP, TJ, NSTAGES, (IP > 3 ? 1 : 2), BODY, PART>;   // 16 targets/thread: one CTA per SM
    const size_t smem = force_sym_smem_bytes<IP, TJ, NSTAGES>();
    static int attr_epoch = 0;
    if (attr_epoch != g.init_epoch) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_epoch = g.init_epoch;
    }
    dim3 grid((unsigned)geo.a_count, (unsigned)geo.splits);
    return launch_ex(kern, grid, dim3(FORCE_THREADS), smem, st, pdl, packed, geo.nb, geo.splits, k_begin, k_count,
                     with_plain, eps2, partials, geo.n_pad, mass_flag, generation, step_ctr, geo.a_begin);
}

// whole evaluations (all nb target blocks) and shares of one (colatus_forces_symmetric_part) are separate instantiations
template <int IP, int TJ, int BODY>
cudaError_t launch_force_sym_body(const Geometry &geo, const float4 *packed, int k_begin, int k_count, int with_plain,
                                  float eps2, float4 *partials, const int *mass_flag, int generation, int *step_ctr,
                                  cudaStream_t st, bool pdl) {
    if (geo.a_begin == 0 && geo.a_count == geo.nb)
        return launch_force_sym_inst<IP, TJ, BODY, false>(geo, packed, k_begin, k_count, with_plain, eps2, partials,
                                                          mass_flag, generation, step_ctr, st, pdl);
    return launch_force_sym_inst<IP, TJ, BODY, true>(geo, packed, k_begin, k_count, with_plain, eps2, partials,
                                                     mass_flag, generation, step_ctr, st, pdl);
}

inline bool sym_pair(const Geometry &geo) { return geo.n_pad >= SYM_PAIR_N; }

cudaError_t launch_force_sym(const Geometry &geo, const float4 *packed, int k_begin, int k_count, int with_plain,
                             float eps2, float4 *partials, const int *mass_flag, int generation, int *step_ctr,
                             cudaStream_t st, bool pdl) {
    if (geo.IP == 2)
        return launch_force_sym_body<2, 256, 0>(geo, packed, k_begin, k_count, with_plain, eps2, partials, mass_flag,
                                                generation, step_ctr, st, pdl);
    if (geo.IP == 3 && !sym_pair(geo))
        return launch_force_sym_body<3, 512, 0>(geo, packed, k_begin, k_count, with_plain, eps2, partials, mass_flag,
                                                generation, step_ctr, st, pdl);
    if (geo.IP == 8 && !sym_pair(geo))
        return launch_force_sym_body<8, 512, 0>(geo, packed, k_begin, k_count, with_plain, eps2, partials, mass_flag,
                                                generation, step_ctr, st, pdl);
    cudaError_t e = geo.IP == 8 ? launch_force_sym_body<8, 512, 1>(geo, packed, k_begin, k_count, with_plain, eps2,
                                                                   partials, mass_flag, generation, step_ctr, st, pdl)
                                : launch_force_sym_body<3, 512, 1>(geo, packed, k_begin, k_count, with_plain, eps2,
                                                                   partials, mass_flag, generation, step_ctr, st, pdl);
    if (e != cudaSuccess) return e;
    g.launches++;
    return geo.IP == 8 ? launch_force_sym_body<8, 512, 2>(geo, packed, k_begin, k_count, with_plain, eps2, partials,
                                                          mass_flag, generation, step_ctr, st, pdl)
                       : launch_force_sym_body<3, 512, 2>(geo, packed, k_begin, k_count, with_plain, eps2, partials,
                                                          mass_flag, generation, step_ctr, st, pdl);
}

// potential evaluations: the 1024-body variant with the fourth (potential) component, both tile bodies in one kernel
cudaError_t launch_force_sym_pot(const Geometry &geo, const float4 *packed, int k_begin, int k_count, int with_plain,
                                 float eps2, float4 *partials, const int *mass_flag, int generation, cudaStream_t st) {
    auto kern = force_sym_pot_kernel<2, 256, NSTAGES, 2>;
    const size_t smem = force_sym_pot_smem_bytes<2, 256, NSTAGES>();
    static int attr_epoch = 0;
    if (attr_epoch != g.init_epoch) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_epoch = g.init_epoch;
    }
    dim3 grid((unsigned)geo.a_count, (unsigned)geo.splits);
    return launch_ex(kern, grid, dim3(FORCE_THREADS), smem, st, false, packed, geo.nb, geo.splits, k_begin, k_count,
                     with_plain, eps2, partials, geo.n_pad, mass_flag, generation);
}

template <int IP, int TJ, bool POT>
cudaError_t launch_force_variant(const Geometry &geo, const float4 *pos_mass, const float4 *packed, int64_t t_begin,
                                 int64_t t_count, float eps2, float scale, int final_out, float4 *out,
                                 int64_t out_stride, const int *mass_flag, int generation, int *step_ctr,
                                 cudaStream_t st, bool pdl) {
    auto kern = force_kernel<IP, TJ, NSTAGES, POT, 2>;
    const size_t smem = force_smem_bytes<IP, TJ, NSTAGES, POT>();
    static int attr_epoch = 0;            // function attributes are per device: set again after every colatus_init
    if (attr_epoch != g.init_epoch) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_epoch = g.init_epoch;
    }
    dim3 grid((unsigned)geo.tiles_t, (unsigned)geo.splits);
    return launch_ex(kern, grid, dim3(FORCE_THREADS), smem, st, pdl, pos_mass, packed, t_begin, t_count,
                     geo.tiles_per_split, eps2, scale, final_out, out, out_stride, mass_flag, generation, step_ctr);
}

template <bool POT>
cudaError_t launch_force(const Geometry &geo, const float4 *pos_mass, const float4 *packed, int64_t t_begin,
                         int64_t t_count, float eps2, float scale, int final_out, float4 *out, int64_t out_stride,
                         const int *mass_flag, int generation, int *step_ctr, cudaStream_t st, bool pdl) {
    switch (geo.IP) {
        case 3:
            return launch_force_variant<3, 512, POT>(geo, pos_mass, packed, t_begin, t_count, eps2, scale,
                                                      final_out, out, out_stride, mass_flag, generation, step_ctr, st, pdl);
        case 2:
            return launch_force_variant<2, 512, POT>(geo, pos_mass, packed, t_begin, t_count, eps2, scale,
                                                     final_out, out, out_stride, mass_flag, generation, step_ctr, st, pdl);
        default:
            return launch_force_variant<1, 128, POT>(geo, pos_mass, packed, t_begin, t_count, eps2, scale,
                                                     final_out, out, out_stride, mass_flag, generation, step_ctr, st, pdl);
    }
}

// colatus_profile: take an event pair from the pool, record the first on `st` now; the caller records *end after the
// last force-kernel launch of the evaluation (left null when profiling is off).
int profile_begin(cudaStream_t st, cudaEvent_t *end) {
    *end = nullptr;
    if (!g.profile) return COLATUS_OK;
    if (g.ev_used + 2 > g.ev_pool.size()) {
        for (int i = 0; i < 64; ++i) {
            cudaEvent_t e;
            CUDA_TRY(cudaEventCreate(&e));
            g.ev_pool.push_back(e);
        }
    }
    cudaEvent_t begin = g.ev_pool[g.ev_used++];
    *end = g.ev_pool[g.ev_used++];
    CUDA_TRY(cudaEventRecord(begin, st));
    return COLATUS_OK;
}

// stage + force (+ reduce): the whole of step a3.  No validation here.
// `fused` (whole-range steps only): the staging pass also applies the drift of eq. (3) to the resident
// positions (drift_stage_kernel), and the partial-sum reduction is left to the caller's fused
// reduce-kick-drift kernel (*deferred_splits = number of partials to add, 0 if `out` is already final).
struct FusedStep {
    StepSrc src;
    int deferred_splits = 0;
    int64_t deferred_stride = 0;   // bodies per partial row
    // two-kernel step loop of colatus_run: the staged array was written by the previous tail/head kernel (no staging
    // launch here), one equal-mass generation stamp serves the whole run, and the force kernel hands the step
    // counter over (force_kernels.cuh)
    bool skip_stage = false;
    int fixed_generation = 0;
    int *step_ctr = nullptr;
    bool pdl = false;          // launch the force kernel as a programmatic dependent of its predecessor
    Geometry geo;              // out: the geometry used (n_pad for the tail/head kernel's grid)
};

// eq. (10) source and mean-density background (colatus_set_deformation / _background): O(n) epilogue on finished
// forces `out` = float4[t_count] of the targets [t_begin, t_begin + t_count).  Nothing is launched when both are off.
int enqueue_external(const float4 *pos_mass, int64_t t_begin, int64_t t_count, float eps2, float4 *out, cudaStream_t st) {
    if (g.def_S == 0.0 && g.bg_rho == 0.0) return COLATUS_OK;
    const double B = (4.0 * 3.14159265358979323846 / 3.0) * g.G * g.bg_rho;
    external_field_kernel<<<(unsigned)((t_count + 255) / 256), 256, 0, st>>>(
        pos_mass, t_begin, t_count, out, (float)g.def_S, (float)g.def_x[0], (float)g.def_x[1], (float)g.def_x[2], eps2,
        (float)B, (float)g.bg_c[0], (float)g.bg_c[1], (float)g.bg_c[2]);
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    return COLATUS_OK;
}

int run_forces(const float4 *pos_mass, int64_t n, int64_t t_begin, int64_t t_count, float eps2, float4 *out,
               bool potential, cudaStream_t st, FusedStep *fused = nullptr) {
    const Workspace w = workspace_layout(n);
    if (w.total > g.ws_bytes)
        return fail(COLATUS_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, n=%lld needs %zu", g.ws_bytes,
                    (long long)n, w.total);
    const Geometry geo = choose_geometry(n, t_count, potential);
    float4 *packed = reinterpret_cast<float4 *>(g.ws + w.packed);
    float4 *partials = reinterpret_cast<float4 *>(g.ws + w.partials);

    // equal-mass detection: a fresh generation per force evaluation; a body whose mass differs from body 0's
    // stamps it into the flag, the force kernel compares (force_kernels.cuh)
    int *mass_flag = reinterpret_cast<int *>(g.ws + Workspace::mass_flag);
    int generation;
    if (fused && fused->fixed_generation) {
        generation = fused->fixed_generation;
    } else {
        g.generation = g.generation == 0x7fffffff ? 1 : g.generation + 1;
        generation = g.generation;
    }
    if (fused) fused->geo = geo;
    if (fused && fused->skip_stage) {
        // staged by the caller's tail/head kernel
    } else {
        if (fused)
            drift_stage_kernel<<<(unsigned)((geo.n_pad + 255) / 256), 256, 0, st>>>(g.pos, g.vel, n, geo.n_pad, packed,
                                                                                    mass_flag, generation, fused->src);
        else
            stage_sources_kernel<<<(unsigned)((geo.n_pad + 255) / 256), 256, 0, st>>>(pos_mass, n, geo.n_pad, packed,
                                                                                      mass_flag, generation);
        CUDA_TRY(cudaGetLastError());
        g.launches++;
    }

    cudaEvent_t e1 = nullptr;                   // colatus_profile: bracket this evaluation's force-kernel launches
    if (int rc = profile_begin(st, &e1)) return rc;
    int *step_ctr = fused ? fused->step_ctr : nullptr;
    if (geo.sym) {
        // every pair once (force_sym_kernels.cuh): one launch per chunk of block distances; its rows (target-side
        // sums of the splits, then one reaction row per distance) are added in row order by the reduction -- inside
        // the caller's fused kick kernel when one launch covers all distances, else here, chunk after chunk into
        // `out` (a fused caller is then told that `out` is final: deferred_splits = 0)
        const unsigned blocks = (unsigned)((n + 255) / 256);
        for (int c = 0; c < geo.chunks; ++c) {
            const int k_begin = 1 + c * geo.K;
            const int k_count = geo.H - c * geo.K < geo.K ? geo.H - c * geo.K : geo.K;
            if (potential)
                CUDA_TRY(launch_force_sym_pot(geo, packed, k_begin, k_count, c == 0, eps2, partials, mass_flag,
                                              generation, st));
            else
                CUDA_TRY(launch_force_sym(geo, packed, k_begin, k_count, c == 0, eps2, partials, mass_flag, generation,
                                          c == 0 ? step_ctr : nullptr, st, fused && fused->pdl && c == 0));
            g.launches++;
            if (fused && geo.chunks == 1) {
                if (g.profile) CUDA_TRY(cudaEventRecord(e1, st));
                fused->deferred_splits = geo.splits + k_count;
                fused->deferred_stride = geo.n_pad;
                return COLATUS_OK;
            }
            if (c == 0 && g.profile && geo.chunks == 1) CUDA_TRY(cudaEventRecord(e1, st));
            if (potential && c == 0)      // the j = k term of the diagonal tiles is removed once, with the first chunk
                reduce_partials_kernel<true, false><<<blocks, 256, 0, st>>>(partials, geo.n_pad, geo.splits + k_count, n,
                                                                            (float)g.G, eps2, pos_mass, 0, out);
            else if (potential)
                reduce_sym_pot_more_kernel<<<blocks, 256, 0, st>>>(partials, geo.n_pad, geo.splits + k_count, n,
                                                                   (float)g.G, out);
            else if (geo.chunks == 1)
                reduce_partials_kernel<false, false><<<blocks, 256, 0, st>>>(partials, geo.n_pad, geo.splits + k_count, n,
                                                                             (float)g.G, eps2, pos_mass, 0, out);
            else {
                // chunked: the chunks' row sums are carried in FP64 (workspace) and rounded once, with the last chunk,
                // so the number of chunks -- the row budget -- does not show in the result's error
                double *acc64 = reinterpret_cast<double *>(g.ws + w.acc64);
                const int rows = geo.splits + k_count;
                if (c == 0)
                    reduce_partials_chunk_kernel<true, false><<<blocks, 256, 0, st>>>(partials, geo.n_pad, rows, n,
                                                                                      (float)g.G, acc64, out);
                else if (c + 1 < geo.chunks)
                    reduce_partials_chunk_kernel<false, false><<<blocks, 256, 0, st>>>(partials, geo.n_pad, rows, n,
                                                                                       (float)g.G, acc64, out);
                else
                    reduce_partials_chunk_kernel<false, true><<<blocks, 256, 0, st>>>(partials, geo.n_pad, rows, n,
                                                                                      (float)g.G, acc64, out);
            }
            CUDA_TRY(cudaGetLastError());
            g.launches++;
        }
        if (g.profile && geo.chunks > 1) CUDA_TRY(cudaEventRecord(e1, st));
        if (fused) {
            fused->deferred_splits = 0;
            fused->deferred_stride = n;
            return COLATUS_OK;
        }
    } else {
        const bool single = geo.splits == 1;
        float4 *fout = single ? out : partials;
        const float scale = single ? (float)g.G : 1.0f;
        cudaError_t e = potential ? launch_force<true>(geo, pos_mass, packed, t_begin, t_count, eps2, scale, single, fout,
                                                       t_count, mass_flag, generation, step_ctr, st, fused && fused->pdl)
                                  : launch_force<false>(geo, pos_mass, packed, t_begin, t_count, eps2, scale, single,
                                                        fout, t_count, mass_flag, generation, step_ctr, st,
                                                        fused && fused->pdl);
        CUDA_TRY(e);
        g.launches++;
        if (g.profile) CUDA_TRY(cudaEventRecord(e1, st));

        if (fused) {
            fused->deferred_splits = single ? 0 : geo.splits;
            fused->deferred_stride = t_count;
            return COLATUS_OK;                      // no external terms in fused steps (checked by the caller)
        }
        if (!single) {
            const unsigned blocks = (unsigned)((t_count + 255) / 256);
            if (potential)
                reduce_partials_kernel<true><<<blocks, 256, 0, st>>>(partials, t_count, geo.splits, t_count, (float)g.G,
                                                                     eps2, pos_mass, t_begin, out);
            else
                reduce_partials_kernel<false><<<blocks, 256, 0, st>>>(partials, t_count, geo.splits, t_count,
                                                                      (float)g.G, eps2, pos_mass, t_begin, out);
            CUDA_TRY(cudaGetLastError());
            g.launches++;
        }
    }
    return enqueue_external(pos_mass, t_begin, t_count, eps2, out, st);
}

// One share of a symmetric evaluation: the block pairs whose target block lies in share `part` of `parts` (contiguous
// block ranges of near-equal length: equal work, the pairing is circulant).  out[n] = G x what those pairs deliver, to
// their target blocks and, as reactions, to the blocks they meet -- 0 where they deliver nothing.  The outputs of all
// shares add up to the whole force.
int run_forces_sym_part(const float4 *pos_mass, int64_t n, float eps2, int part, int parts, float4 *out,
                        cudaStream_t st) {
    const Workspace w = workspace_layout(n);
    if (w.total > g.ws_bytes)
        return fail(COLATUS_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, n=%lld needs %zu", g.ws_bytes,
                    (long long)n, w.total);
    const Geometry geo = choose_sym_geometry(n, part, parts);
    if (!geo.sym) return fail(COLATUS_INVALID_ARG, "n=%lld is too small for a symmetric evaluation", (long long)n);
    float4 *packed = reinterpret_cast<float4 *>(g.ws + w.packed);
    float4 *partials = reinterpret_cast<float4 *>(g.ws + w.partials);
    int *mass_flag = reinterpret_cast<int *>(g.ws + Workspace::mass_flag);
    g.generation = g.generation == 0x7fffffff ? 1 : g.generation + 1;
    const int generation = g.generation;
    stage_sources_kernel<<<(unsigned)((geo.n_pad + 255) / 256), 256, 0, st>>>(pos_mass, n, geo.n_pad, packed, mass_flag,
                                                                              generation);
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    if (geo.a_count == 0) {                      // more shares than blocks: this share delivers nothing
        CUDA_TRY(cudaMemsetAsync(out, 0, (size_t)n * 16, st));
        return COLATUS_OK;
    }
    cudaEvent_t e1 = nullptr;                   // colatus_profile: bracket this evaluation's force-kernel launches
    if (int rc = profile_begin(st, &e1)) return rc;
    for (int c = 0; c < geo.chunks; ++c) {
        const int k_begin = 1 + c * geo.K;
        const int k_count = geo.H - c * geo.K < geo.K ? geo.H - c * geo.K : geo.K;
        CUDA_TRY(launch_force_sym(geo, packed, k_begin, k_count, c == 0, eps2, partials, mass_flag, generation, nullptr,
                                  st, false));
        g.launches++;
        if (g.profile && c == 0 && geo.chunks == 1) CUDA_TRY(cudaEventRecord(e1, st));
        if (c == 0)
            reduce_sym_part_kernel<false><<<blocks, 256, 0, st>>>(partials, geo.n_pad, geo.splits, k_begin, k_count,
                                                                  geo.nb, (int)geo.bt(), geo.a_begin, geo.a_count, 1, n,
                                                                  (float)g.G, out);
        else
            reduce_sym_part_kernel<true><<<blocks, 256, 0, st>>>(partials, geo.n_pad, geo.splits, k_begin, k_count,
                                                                 geo.nb, (int)geo.bt(), geo.a_begin, geo.a_count, 0, n,
                                                                 (float)g.G, out);
        CUDA_TRY(cudaGetLastError());
        g.launches++;
    }
    if (g.profile && geo.chunks > 1) CUDA_TRY(cudaEventRecord(e1, st));
    return COLATUS_OK;
}

// The branch-free self term (reading G4) is exactly 0 only while w = m_k rinv^3 stays finite in FP32 (0 * inf = NaN):
// rinv^3 = eps2^-1.5 <= 1e36 at this floor, which leaves masses up to ~3e2 in magnitude (colatus.h "eps2").
inline bool eps2_ok(float eps2) { return std::isfinite(eps2) && eps2 >= 1e-24f; }

int check_forces_args(const void *pos_mass, int64_t n, int64_t t_begin, int64_t t_count, float eps2,
                      const void *acc_out) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!pos_mass || !acc_out) return fail(COLATUS_INVALID_ARG, "null pointer");
    if (n < 1 || n > 2147483647LL) return fail(COLATUS_INVALID_ARG, "n=%lld out of [1, 2^31-1]", (long long)n);
    if (t_begin < 0 || t_count < 1 || t_begin + t_count > n)
        return fail(COLATUS_INVALID_ARG, "target range [%lld, +%lld) outside [0, %lld)", (long long)t_begin,
                    (long long)t_count, (long long)n);
    if (!aligned16(pos_mass) || !aligned16(acc_out)) return fail(COLATUS_INVALID_ARG, "pointer not 16-byte aligned");
    if (pos_mass == acc_out) return fail(COLATUS_INVALID_ARG, "pos_mass and acc_out alias");
    if (!eps2_ok(eps2)) return fail(COLATUS_INVALID_ARG, "eps2 must be finite and >= 1e-24");
    return COLATUS_OK;
}

int enqueue_drift(double d) {
    const unsigned blocks = (unsigned)((g.t_count + 255) / 256);
    drift_kernel<<<blocks, 256, 0, g.stream>>>(g.pos, g.vel, g.t_begin, g.t_count, (float)d);
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    return COLATUS_OK;
}

// eqs. (4)-(5) for the target range from forces in `acc` (float4[t_count], indexed from the range's first body)
int enqueue_kick_drift(const float4 *acc, double cv, double ck, double d2, float tag) {
    const unsigned blocks = (unsigned)((g.t_count + 255) / 256);
    if (g.trace_k > 0) {
        const Workspace w = workspace_layout(g.n);
        const int32_t *slot = reinterpret_cast<const int32_t *>(g.ws + w.trace_slot);
        float4 *row = g.ring + (size_t)(g.step % g.trace_cap) * g.trace_k;
        kick_drift_kernel<true><<<blocks, 256, 0, g.stream>>>(g.pos, g.vel, acc, g.t_begin, g.t_count, (float)cv,
                                                              (float)ck, (float)d2, slot, row, tag);
    } else {
        kick_drift_kernel<false><<<blocks, 256, 0, g.stream>>>(g.pos, g.vel, acc, g.t_begin, g.t_count, (float)cv,
                                                               (float)ck, (float)d2, nullptr, nullptr, tag);
    }
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    g.step++;
    return COLATUS_OK;
}

int enqueue_force_kick_drift(double cv, double ck, double d2, float tag) {
    int rc = run_forces(g.pos, g.n, g.t_begin, g.t_count, g.eps2, g.acc, false, g.stream);
    if (rc) return rc;
    return enqueue_kick_drift(g.acc, cv, ck, d2, tag);
}

// Whole-range step without external terms: three launches (drift+stage, force, reduce+kick+drift).
bool can_fuse_step() { return g.t_begin == 0 && g.t_count == g.n && g.def_S == 0.0 && g.bg_rho == 0.0; }

int enqueue_step_fused(StepSrc src, cudaStream_t st) {
    FusedStep f;
    f.src = src;
    if (g.trace_k > 0 && !src.table) f.src.ring_row = (int)(g.step % g.trace_cap);
    int rc = run_forces(g.pos, g.n, 0, g.n, g.eps2, g.acc, false, st, &f);
    if (rc) return rc;
    const Workspace w = workspace_layout(g.n);
    const unsigned blocks = (unsigned)((g.n + 255) / 256);
    const int32_t *slot = reinterpret_cast<const int32_t *>(g.ws + w.trace_slot);
    const float4 *partials = reinterpret_cast<const float4 *>(g.ws + w.partials);
    if (f.deferred_splits > 0) {
        if (g.trace_k > 0)
            reduce_kick_drift_kernel<true><<<blocks, 256, 0, st>>>(g.pos, g.vel, g.acc, partials, f.deferred_stride,
                                                                   f.deferred_splits, g.n, (float)g.G, f.src, slot, g.ring,
                                                                   g.trace_k);
        else
            reduce_kick_drift_kernel<false><<<blocks, 256, 0, st>>>(g.pos, g.vel, g.acc, partials, f.deferred_stride,
                                                                    f.deferred_splits, g.n, (float)g.G, f.src, nullptr,
                                                                    nullptr, 0);
    } else if (src.table) {                      // single split: acc is final, plain kick-drift
        if (g.trace_k > 0)
            kick_drift_table_kernel<true><<<blocks, 256, 0, st>>>(g.pos, g.vel, g.acc, 0, g.n, src.table, src.ctr, slot,
                                                                  g.ring, g.trace_k);
        else
            kick_drift_table_kernel<false><<<blocks, 256, 0, st>>>(g.pos, g.vel, g.acc, 0, g.n, src.table, src.ctr,
                                                                   nullptr, nullptr, 0);
    } else {
        float4 *row = g.trace_k > 0 ? g.ring + (size_t)f.src.ring_row * g.trace_k : nullptr;
        if (g.trace_k > 0)
            kick_drift_kernel<true><<<blocks, 256, 0, st>>>(g.pos, g.vel, g.acc, 0, g.n, src.cv, src.ck, src.d2, slot,
                                                            row, src.tag);
        else
            kick_drift_kernel<false><<<blocks, 256, 0, st>>>(g.pos, g.vel, g.acc, 0, g.n, src.cv, src.ck, src.d2,
                                                             nullptr, nullptr, src.tag);
    }
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    return COLATUS_OK;
}

// One step with scalar coefficients on the resident stream: fused when possible, else the five launches.
int enqueue_step_scalar(double d1, double cv, double ck, double d2, float tag) {
    if (can_fuse_step()) {
        StepSrc src{nullptr, nullptr, (float)d1, (float)cv, (float)ck, (float)d2, tag, 0};
        int rc = enqueue_step_fused(src, g.stream);
        if (rc == COLATUS_OK) g.step++;
        return rc;
    }
    int rc = enqueue_drift(d1);
    if (rc) return rc;
    return enqueue_force_kick_drift(cv, ck, d2, tag);
}

void invalidate_graph() { g.graph_valid = false; }   // both graphs are rebuilt at the next colatus_run

// One step with the coefficients of table row ctr[0] (integrate_kernels.cuh "table-driven variants"):
// the same launches as colatus_step (fused when possible), with step-independent arguments, on stream `st`.
int enqueue_step_table(cudaStream_t st) {
    const Workspace w = workspace_layout(g.n);
    const StepCoef *table = reinterpret_cast<const StepCoef *>(g.ws + w.step_table);
    int *ctr = reinterpret_cast<int *>(g.ws + w.step_ctr);
    if (can_fuse_step()) {
        StepSrc src{table, ctr, 0.f, 0.f, 0.f, 0.f, 0.f, 0};
        return enqueue_step_fused(src, st);
    }
    const unsigned blocks = (unsigned)((g.t_count + 255) / 256);
    drift_table_kernel<<<blocks, 256, 0, st>>>(g.pos, g.vel, g.t_begin, g.t_count, table, ctr);
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    int rc = run_forces(g.pos, g.n, g.t_begin, g.t_count, g.eps2, g.acc, false, st);
    if (rc) return rc;
    if (g.trace_k > 0) {
        const int32_t *slot = reinterpret_cast<const int32_t *>(g.ws + w.trace_slot);
        kick_drift_table_kernel<true><<<blocks, 256, 0, st>>>(g.pos, g.vel, g.acc, g.t_begin, g.t_count, table, ctr,
                                                              slot, g.ring, g.trace_k);
    } else {
        kick_drift_table_kernel<false><<<blocks, 256, 0, st>>>(g.pos, g.vel, g.acc, g.t_begin, g.t_count, table, ctr,
                                                               nullptr, nullptr, 0);
    }
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    return COLATUS_OK;
}

// ---- two-kernel step loop of colatus_run (whole range, no external terms; integrate_kernels.cuh) --------------
// head: the first half drift + staging of the run's first step (row ctr[0] of the table);
// step: force kernel (+ step-counter hand-over) and the tail/head kernel.  `generation` is one equal-mass stamp
// for the whole run (a captured graph keeps replaying the same value).
int enqueue_run_head(cudaStream_t st, int generation) {
    const Workspace w = workspace_layout(g.n);
    const Geometry geo = choose_geometry(g.n, g.n);
    const StepCoef *table = reinterpret_cast<const StepCoef *>(g.ws + w.step_table);
    int *ctr = reinterpret_cast<int *>(g.ws + w.step_ctr);
    float4 *packed = reinterpret_cast<float4 *>(g.ws + w.packed);
    int *mass_flag = reinterpret_cast<int *>(g.ws + Workspace::mass_flag);
    StepSrc src{table, ctr, 0.f, 0.f, 0.f, 0.f, 0.f, 0};
    drift_stage_kernel<<<(unsigned)((geo.n_pad + 255) / 256), 256, 0, st>>>(g.pos, g.vel, g.n, geo.n_pad, packed, mass_flag,
                                                                            generation, src);
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    return COLATUS_OK;
}

int enqueue_step_two_kernels(cudaStream_t st, int generation) {
    const Workspace w = workspace_layout(g.n);
    const StepCoef *table = reinterpret_cast<const StepCoef *>(g.ws + w.step_table);
    int *ctr = reinterpret_cast<int *>(g.ws + w.step_ctr);
    FusedStep f;
    f.skip_stage = true;
    f.fixed_generation = generation;
    f.step_ctr = ctr;
    f.pdl = true;
    int rc = run_forces(g.pos, g.n, 0, g.n, g.eps2, g.acc, false, st, &f);
    if (rc) return rc;
    const unsigned blocks = (unsigned)((f.geo.n_pad + COLATUS_TAIL_THREADS - 1) / COLATUS_TAIL_THREADS);
    const int32_t *slot = reinterpret_cast<const int32_t *>(g.ws + w.trace_slot);
    const float4 *partials = reinterpret_cast<const float4 *>(g.ws + w.partials);
    float4 *packed = reinterpret_cast<float4 *>(g.ws + w.packed);
    int *mass_flag = reinterpret_cast<int *>(g.ws + Workspace::mass_flag);
    cudaError_t e;
    if (g.trace_k > 0)
        e = launch_ex(step_tail_head_kernel<true>, dim3(blocks), dim3(COLATUS_TAIL_THREADS), 0, st, true, g.pos, g.vel, g.acc, partials,
                      f.deferred_stride, f.deferred_splits, g.n, f.geo.n_pad, (float)g.G, table, ctr, slot, g.ring, g.trace_k, packed,
                      mass_flag, generation);
    else
        e = launch_ex(step_tail_head_kernel<false>, dim3(blocks), dim3(COLATUS_TAIL_THREADS), 0, st, true, g.pos, g.vel, g.acc, partials,
                      f.deferred_stride, f.deferred_splits, g.n, f.geo.n_pad, (float)g.G, table, ctr, (const int32_t *)nullptr,
                      (float4 *)nullptr, 0, packed, mass_flag, generation);
    CUDA_TRY(e);
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    return COLATUS_OK;
}

int build_trace_map(const int32_t *idx_dev) {
    const Workspace w = workspace_layout(g.n);
    if (w.total > g.ws_bytes) return fail(COLATUS_WORKSPACE_TOO_SMALL, "workspace too small for n=%lld", (long long)g.n);
    int32_t *slot = reinterpret_cast<int32_t *>(g.ws + w.trace_slot);
    trace_fill_kernel<<<(unsigned)((g.n + 255) / 256), 256, 0, g.stream>>>(slot, g.n);
    CUDA_TRY(cudaGetLastError());
    trace_scatter_kernel<<<(unsigned)((g.trace_k + 255) / 256), 256, 0, g.stream>>>(slot, g.n, idx_dev, g.trace_k);
    CUDA_TRY(cudaGetLastError());
    g.launches += 2;
    return COLATUS_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

size_t colatus_workspace_bytes(int64_t n_max) {
    if (n_max < 1) return 0;
    return workspace_layout(n_max).total;
}

int colatus_init(const colatus_config *cfg) {
    if (g.initialised) return fail(COLATUS_ALREADY_INITIALISED, "colatus_init called twice without colatus_shutdown");
    if (!cfg) return fail(COLATUS_INVALID_ARG, "cfg is null");
    if (!std::isfinite(cfg->G)) return fail(COLATUS_INVALID_ARG, "G is not finite");
    if (!cfg->workspace_dev || (reinterpret_cast<uintptr_t>(cfg->workspace_dev) & 255u))
        return fail(COLATUS_INVALID_ARG, "workspace_dev is null or not 256-byte aligned");
    CUDA_TRY(cudaSetDevice(cfg->device));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, cfg->device));
    if (prop.major != 10)
        return fail(COLATUS_UNSUPPORTED_DEVICE, "device %d (%s) is cc %d.%d; libcolatus is built for sm_100a only",
                    cfg->device, prop.name, prop.major, prop.minor);
    g.G = cfg->G;
    g.device = cfg->device;
    g.sm_count = prop.multiProcessorCount;
    g.ctas_per_sm = 2;
    if (cfg->workspace_bytes < 256) return fail(COLATUS_WORKSPACE_TOO_SMALL, "workspace smaller than 256 bytes");
    CUDA_TRY(cudaMemset(cfg->workspace_dev, 0, 256));        // mass_flag and friends
    g.ws = static_cast<unsigned char *>(cfg->workspace_dev);
    g.ws_bytes = cfg->workspace_bytes;
    g.generation = 0;
    g.init_epoch++;
    g.uploaded = false;
    g.trace_k = 0;
    g.step = 0;
    g.profile = false;
    g.ev_used = 0;
    g.force_I = g.force_splits = 0;
    g.symmetric = 1;
    g.sym_rows = 0;
    g.sym_block = 0;
    g.def_S = g.bg_rho = 0.0;
    invalidate_graph();
    g.initialised = true;
    g.err[0] = 0;
    return COLATUS_OK;
}

void colatus_shutdown(void) {
    if (g.graph_exec) cudaGraphExecDestroy(g.graph_exec);
    if (g.graph) cudaGraphDestroy(g.graph);
    if (g.graph_exec_k) cudaGraphExecDestroy(g.graph_exec_k);
    if (g.graph_k) cudaGraphDestroy(g.graph_k);
    g.graph_exec_k = nullptr;
    g.graph_k = nullptr;
    if (g.run_ev_in) cudaEventDestroy(g.run_ev_in);
    if (g.run_ev_out) cudaEventDestroy(g.run_ev_out);
    if (g.run_stream) cudaStreamDestroy(g.run_stream);
    g.graph_exec = nullptr;
    g.graph = nullptr;
    g.run_ev_in = g.run_ev_out = nullptr;
    g.run_stream = nullptr;
    g.graph_valid = false;
    for (cudaEvent_t e : g.ev_pool) cudaEventDestroy(e);
    g.ev_pool.clear();
    g.ev_used = 0;
    g.initialised = false;
    g.uploaded = false;
    g.trace_k = 0;
    g.ws = nullptr;
    g.ws_bytes = 0;
}

int colatus_forces(const void *pos_mass_dev, int64_t n, float eps2, void *acc_out_dev, void *cuda_stream) {
    int rc = check_forces_args(pos_mass_dev, n, 0, n, eps2, acc_out_dev);
    if (rc) return rc;
    return run_forces(static_cast<const float4 *>(pos_mass_dev), n, 0, n, eps2, static_cast<float4 *>(acc_out_dev),
                      false, static_cast<cudaStream_t>(cuda_stream));
}

int colatus_forces_potential(const void *pos_mass_dev, int64_t n, float eps2, void *acc_out_dev, void *cuda_stream) {
    int rc = check_forces_args(pos_mass_dev, n, 0, n, eps2, acc_out_dev);
    if (rc) return rc;
    return run_forces(static_cast<const float4 *>(pos_mass_dev), n, 0, n, eps2, static_cast<float4 *>(acc_out_dev),
                      true, static_cast<cudaStream_t>(cuda_stream));
}

int colatus_forces_range(const void *pos_mass_dev, int64_t n, int64_t target_begin, int64_t target_count, float eps2,
                         void *acc_out_dev, void *cuda_stream) {
    int rc = check_forces_args(pos_mass_dev, n, target_begin, target_count, eps2, acc_out_dev);
    if (rc) return rc;
    return run_forces(static_cast<const float4 *>(pos_mass_dev), n, target_begin, target_count, eps2,
                      static_cast<float4 *>(acc_out_dev), false, static_cast<cudaStream_t>(cuda_stream));
}

int colatus_forces_symmetric_part(const void *pos_mass_dev, int64_t n, float eps2, int part, int parts,
                                  void *acc_out_dev, void *cuda_stream) {
    int rc = check_forces_args(pos_mass_dev, n, 0, n, eps2, acc_out_dev);
    if (rc) return rc;
    if (parts < 1 || part < 0 || part >= parts) return fail(COLATUS_INVALID_ARG, "need 0 <= part < parts");
    return run_forces_sym_part(static_cast<const float4 *>(pos_mass_dev), n, eps2, part, parts,
                               static_cast<float4 *>(acc_out_dev), static_cast<cudaStream_t>(cuda_stream));
}

int colatus_forces_host(const float *pos_mass_host, int64_t n, float eps2, float *acc_out_host, void *cuda_stream) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!pos_mass_host || !acc_out_host) return fail(COLATUS_INVALID_ARG, "null pointer");
    if (n < 1 || n > 2147483647LL) return fail(COLATUS_INVALID_ARG, "n=%lld out of [1, 2^31-1]", (long long)n);
    if (!eps2_ok(eps2)) return fail(COLATUS_INVALID_ARG, "eps2 must be finite and >= 1e-24");
    const Workspace w = workspace_layout(n);
    if (w.total > g.ws_bytes)
        return fail(COLATUS_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, n=%lld needs %zu", g.ws_bytes,
                    (long long)n, w.total);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    float4 *din = reinterpret_cast<float4 *>(g.ws + w.stage_in);
    float4 *dout = reinterpret_cast<float4 *>(g.ws + w.stage_out);
    CUDA_TRY(cudaMemcpyAsync(din, pos_mass_host, (size_t)n * 16, cudaMemcpyHostToDevice, st));
    int rc = run_forces(din, n, 0, n, eps2, dout, false, st);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(acc_out_host, dout, (size_t)n * 16, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return COLATUS_OK;
}

int colatus_upload(void *pos_mass_dev, void *vel_dev, void *acc_dev, int64_t n, float eps2, void *cuda_stream) {
    int rc = check_forces_args(pos_mass_dev, n, 0, n, eps2, acc_dev);
    if (rc) return rc;
    if (!vel_dev || !aligned16(vel_dev)) return fail(COLATUS_INVALID_ARG, "vel_dev null or misaligned");
    if (vel_dev == pos_mass_dev || vel_dev == acc_dev) return fail(COLATUS_INVALID_ARG, "state buffers alias");
    if (workspace_layout(n).total > g.ws_bytes)
        return fail(COLATUS_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, n=%lld needs %zu", g.ws_bytes,
                    (long long)n, workspace_layout(n).total);
    g.pos = static_cast<float4 *>(pos_mass_dev);
    g.vel = static_cast<float4 *>(vel_dev);
    g.acc = static_cast<float4 *>(acc_dev);
    g.n = n;
    g.t_begin = 0;
    g.t_count = n;
    g.eps2 = eps2;
    g.stream = static_cast<cudaStream_t>(cuda_stream);
    g.step = 0;
    g.trace_k = 0;
    g.uploaded = true;
    invalidate_graph();
    return COLATUS_OK;
}

int colatus_set_target_range(int64_t target_begin, int64_t target_count) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    if (target_begin < 0 || target_count < 1 || target_begin + target_count > g.n)
        return fail(COLATUS_INVALID_ARG, "target range outside [0, n)");
    g.t_begin = target_begin;
    invalidate_graph();
    g.t_count = target_count;
    return COLATUS_OK;
}

int colatus_step_coeffs(double d1, double cv, double ck, double d2) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    if (!std::isfinite(d1) || !std::isfinite(cv) || !std::isfinite(ck) || !std::isfinite(d2))
        return fail(COLATUS_INVALID_ARG, "non-finite step coefficient");
    return enqueue_step_scalar(d1, cv, ck, d2, 0.f);
}

int colatus_step_coefficients(double tau, double a, double H, double out[4]) {
    if (!out) return fail(COLATUS_INVALID_ARG, "out is null");
    if (!std::isfinite(tau) || !std::isfinite(a) || !std::isfinite(H))
        return fail(COLATUS_INVALID_ARG, "non-finite tau, a or H");
    if (!(a > 0.0)) return fail(COLATUS_INVALID_ARG, "a must be > 0");
    if (!(1.0 + H * tau > 0.0)) return fail(COLATUS_INVALID_ARG, "1 + H tau must be > 0");
    out[0] = 0.5 * tau;                                   // eq. (3)
    out[1] = (1.0 - H * tau) / (1.0 + H * tau);           // eq. (4): drag factor
    out[2] = tau / (a * a * a * (1.0 + H * tau));         // eq. (4): kick coefficient (a^-3 applied here, G5)
    out[3] = 0.5 * tau;                                   // eq. (5)
    return COLATUS_OK;
}

int colatus_step(double tau, double a, double H) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    double c[4];
    int rc = colatus_step_coefficients(tau, a, H, c);
    if (rc) return rc;
    return enqueue_step_scalar(c[0], c[1], c[2], c[3], (float)a);        // eqs. (3), (1), (4), (5)
}

int colatus_symplectic_coefficients(const colatus_cosmo *c, double a0, double tau, double out[5]) {
    if (!c || !out) return fail(COLATUS_INVALID_ARG, "null pointer");
    if (!std::isfinite(a0) || !(a0 > 0.0) || !std::isfinite(tau)) return fail(COLATUS_INVALID_ARG, "a0 must be > 0, tau finite");
    // eq. (9), PAPER.md:64 (reading G11): drift integrals of dt/a^2 over each half step, kick integral of dt/a
    const double a_mid = colatus_a_advance(c, a0, 0.5 * tau);
    out[0] = colatus_int_dt_over_a_pow(c, a0, 0.5 * tau, 2.0);
    out[1] = 1.0;
    out[2] = colatus_int_dt_over_a_pow(c, a0, tau, 1.0);
    out[3] = colatus_int_dt_over_a_pow(c, a_mid, 0.5 * tau, 2.0);
    out[4] = colatus_a_advance(c, a_mid, 0.5 * tau);
    for (int i = 0; i < 5; ++i)
        if (!std::isfinite(out[i])) return fail(COLATUS_INVALID_ARG, "scale-factor integration failed (a reached 0?)");
    return COLATUS_OK;
}

int colatus_step_symplectic(const colatus_cosmo *c, double a0, double tau, double *a_end) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    double k[5];
    int rc = colatus_symplectic_coefficients(c, a0, tau, k);
    if (rc) return rc;
    rc = enqueue_step_scalar(k[0], k[1], k[2], k[3], (float)k[4]);
    if (rc) return rc;
    if (a_end) *a_end = k[4];
    return COLATUS_OK;
}

int colatus_set_deformation(const double x_psi[3], double strength) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!std::isfinite(strength)) return fail(COLATUS_INVALID_ARG, "strength is not finite");
    if (strength != 0.0) {
        if (!x_psi) return fail(COLATUS_INVALID_ARG, "x_psi is null");
        for (int i = 0; i < 3; ++i)
            if (!std::isfinite(x_psi[i])) return fail(COLATUS_INVALID_ARG, "x_psi is not finite");
        for (int i = 0; i < 3; ++i) g.def_x[i] = x_psi[i];
    }
    g.def_S = strength;
    invalidate_graph();
    return COLATUS_OK;
}

int colatus_set_background(const double centre[3], double rho_bar) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!std::isfinite(rho_bar)) return fail(COLATUS_INVALID_ARG, "rho_bar is not finite");
    if (rho_bar != 0.0) {
        if (!centre) return fail(COLATUS_INVALID_ARG, "centre is null");
        for (int i = 0; i < 3; ++i)
            if (!std::isfinite(centre[i])) return fail(COLATUS_INVALID_ARG, "centre is not finite");
        for (int i = 0; i < 3; ++i) g.bg_c[i] = centre[i];
    }
    g.bg_rho = rho_bar;
    invalidate_graph();
    return COLATUS_OK;
}

static int run_steps(const colatus_cosmo *c, double a_start, double tau, int64_t n_steps, int use_graph, double *a_end,
                     bool symplectic) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    if (n_steps < 1) return fail(COLATUS_INVALID_ARG, "n_steps < 1");
    if (!std::isfinite(tau)) return fail(COLATUS_INVALID_ARG, "tau is not finite");
    if (c && (!std::isfinite(a_start) || !(a_start > 0.0))) return fail(COLATUS_INVALID_ARG, "a_start must be > 0");
    const Workspace w = workspace_layout(g.n);
    if (w.total > g.ws_bytes) return fail(COLATUS_WORKSPACE_TOO_SMALL, "workspace too small for n=%lld", (long long)g.n);

    // the whole schedule first (eq. (2), host, double): nothing is enqueued if any step is invalid
    std::vector<StepCoef> coef((size_t)n_steps);
    double a = c ? a_start : 1.0;
    for (int64_t s = 0; s < n_steps; ++s) {
        double k[4], tag;
        if (symplectic && c) {                               // eq. (9): drift / kick integrals along eq. (2)
            double q[5];
            int rc = colatus_symplectic_coefficients(c, a, tau, q);
            if (rc) return rc;
            k[0] = q[0]; k[1] = q[1]; k[2] = q[2]; k[3] = q[3];
            a = q[4];
            tag = a;                                         // a(t + tau), as colatus_step_symplectic
        } else {
            double a_mid = 1.0, H_mid = 0.0;                 // c == NULL: static background (reading G13)
            if (c) {
                a_mid = colatus_a_advance(c, a, 0.5 * tau);  // a, H at t_n + tau/2 (reading G3)
                H_mid = colatus_hubble(c, a_mid);
                a = colatus_a_advance(c, a_mid, 0.5 * tau);
            }
            int rc = colatus_step_coefficients(tau, a_mid, H_mid, k);
            if (rc) return rc;
            tag = a_mid;
        }
        StepCoef &q = coef[(size_t)s];
        q.d1 = (float)k[0];
        q.cv = (float)k[1];
        q.ck = (float)k[2];
        q.d2 = (float)k[3];
        q.tag = (float)tag;
        q.ring_row = g.trace_k > 0 ? (int)((g.step + s) % g.trace_cap) : 0;
        q.d1_next = 0.f;
        q.has_next = 0;
        if (s > 0) {                                         // two-kernel loop: the tail of step s-1 does this step's head
            coef[(size_t)s - 1].d1_next = q.d1;
            coef[(size_t)s - 1].has_next = 1;
        }
    }

    if (!g.run_stream) {
        CUDA_TRY(cudaStreamCreateWithFlags(&g.run_stream, cudaStreamNonBlocking));
        CUDA_TRY(cudaEventCreateWithFlags(&g.run_ev_in, cudaEventDisableTiming));
        CUDA_TRY(cudaEventCreateWithFlags(&g.run_ev_out, cudaEventDisableTiming));
    }
    // the loop runs on the library's own stream (the caller's may be the legacy default stream, which
    // cannot be captured), ordered after and before the resident stream by events
    CUDA_TRY(cudaEventRecord(g.run_ev_in, g.stream));
    CUDA_TRY(cudaStreamWaitEvent(g.run_stream, g.run_ev_in, 0));

    const bool profile_was = g.profile;
    g.profile = false;                                      // no event brackets inside a graph
    int rc = COLATUS_OK;
    // whole-range runs without external terms take the two-kernel loop (force + tail/head per step, one head
    // kernel per run); otherwise a step is drift / force (+ reduce, external terms) / kick-drift
    const bool two = can_fuse_step();
    int run_generation = 0;
    if (two && !use_graph) {
        g.generation = g.generation == 0x7fffffff ? 1 : g.generation + 1;
        run_generation = g.generation;
    }
    if (use_graph && !g.graph_valid) {
        if (g.graph_exec) cudaGraphExecDestroy(g.graph_exec);
        if (g.graph) cudaGraphDestroy(g.graph);
        if (g.graph_exec_k) cudaGraphExecDestroy(g.graph_exec_k);
        if (g.graph_k) cudaGraphDestroy(g.graph_k);
        g.graph_exec = g.graph_exec_k = nullptr;
        g.graph = g.graph_k = nullptr;
        g.generation = g.generation == 0x7fffffff ? 1 : g.generation + 1;
        g.graph_generation = g.generation;                  // the captured kernels keep stamping / comparing this value
        // a one-step graph, and for the two-kernel loop also a graph of GRAPH_STEPS consecutive steps (the step
        // index lives on the device, so every step's nodes are identical): replaying several steps at once
        // removes the gap between graph launches, which at N = 4096 is a quarter of a step
        for (int pass = 0; pass < (two ? 2 : 1) && rc == COLATUS_OK; ++pass) {
            cudaGraph_t *gr = pass ? &g.graph_k : &g.graph;
            cudaGraphExec_t *ge = pass ? &g.graph_exec_k : &g.graph_exec;
            cudaError_t e = cudaStreamBeginCapture(g.run_stream, cudaStreamCaptureModeThreadLocal);
            if (e == cudaSuccess) {
                const int64_t launches0 = g.launches;
                for (int k = 0; k < (pass ? GRAPH_STEPS : 1) && rc == COLATUS_OK; ++k)
                    rc = two ? enqueue_step_two_kernels(g.run_stream, g.graph_generation) : enqueue_step_table(g.run_stream);
                if (!pass) g.graph_launches = g.launches - launches0;      // kernels per step
                g.launches = launches0;                                    // captured, not launched
                e = cudaStreamEndCapture(g.run_stream, gr);
                if (rc == COLATUS_OK && e == cudaSuccess) e = cudaGraphInstantiate(ge, *gr, 0);
            }
            if (rc == COLATUS_OK && e != cudaSuccess)
                rc = fail(COLATUS_CUDA_ERROR, "graph capture failed: %s", cudaGetErrorString(e));
        }
        g.graph_valid = rc == COLATUS_OK;
    }
    if (use_graph) run_generation = g.graph_generation;
    StepCoef *table = reinterpret_cast<StepCoef *>(g.ws + w.step_table);
    int *ctr = reinterpret_cast<int *>(g.ws + w.step_ctr);
    for (int64_t s0 = 0; rc == COLATUS_OK && s0 < n_steps; s0 += RUN_CHUNK) {
        const int64_t m = n_steps - s0 < RUN_CHUNK ? n_steps - s0 : RUN_CHUNK;
        cudaError_t e = cudaMemcpyAsync(table, coef.data() + s0, (size_t)m * sizeof(StepCoef), cudaMemcpyHostToDevice,
                                        g.run_stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(ctr, 0, 2 * sizeof(int), g.run_stream);
        if (e != cudaSuccess) {
            rc = fail(COLATUS_CUDA_ERROR, "table upload failed: %s", cudaGetErrorString(e));
            break;
        }
        if (two && s0 == 0) rc = enqueue_run_head(g.run_stream, run_generation);   // later heads ride in the tails
        for (int64_t s = 0; s < m && rc == COLATUS_OK;) {
            int64_t done = 1;
            if (use_graph) {
                const bool multi = g.graph_exec_k && m - s >= GRAPH_STEPS;
                if (multi) done = GRAPH_STEPS;
                e = cudaGraphLaunch(multi ? g.graph_exec_k : g.graph_exec, g.run_stream);
                if (e != cudaSuccess) rc = fail(COLATUS_CUDA_ERROR, "cudaGraphLaunch failed: %s", cudaGetErrorString(e));
                g.launches += g.graph_launches * done;
            } else {
                rc = two ? enqueue_step_two_kernels(g.run_stream, run_generation) : enqueue_step_table(g.run_stream);
            }
            if (rc == COLATUS_OK) g.step += done;
            s += done;
        }
    }
    g.profile = profile_was;
    // the resident stream waits for the loop whatever happened above, so later calls stay ordered
    cudaEventRecord(g.run_ev_out, g.run_stream);
    cudaStreamWaitEvent(g.stream, g.run_ev_out, 0);
    if (rc == COLATUS_OK && a_end) *a_end = a;
    return rc;
}

int colatus_run(const colatus_cosmo *c, double a_start, double tau, int64_t n_steps, int use_graph, double *a_end) {
    return run_steps(c, a_start, tau, n_steps, use_graph, a_end, false);
}

int colatus_run_symplectic(const colatus_cosmo *c, double a_start, double tau, int64_t n_steps, int use_graph,
                           double *a_end) {
    return run_steps(c, a_start, tau, n_steps, use_graph, a_end, true);
}

int colatus_drift(double d) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    if (!std::isfinite(d)) return fail(COLATUS_INVALID_ARG, "non-finite drift coefficient");
    return enqueue_drift(d);
}

int colatus_force_kick_drift(double cv, double ck, double d2) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    if (!std::isfinite(cv) || !std::isfinite(ck) || !std::isfinite(d2))
        return fail(COLATUS_INVALID_ARG, "non-finite step coefficient");
    return enqueue_force_kick_drift(cv, ck, d2, 0.f);
}

int colatus_kick_drift(const void *acc_dev, double cv, double ck, double d2) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    if (!acc_dev || !aligned16(acc_dev)) return fail(COLATUS_INVALID_ARG, "acc_dev null or misaligned");
    if (!std::isfinite(cv) || !std::isfinite(ck) || !std::isfinite(d2))
        return fail(COLATUS_INVALID_ARG, "non-finite step coefficient");
    return enqueue_kick_drift(static_cast<const float4 *>(acc_dev), cv, ck, d2, 0.f);
}

int colatus_add_external(void *acc_dev) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    if (!acc_dev || !aligned16(acc_dev)) return fail(COLATUS_INVALID_ARG, "acc_dev null or misaligned");
    return enqueue_external(g.pos, g.t_begin, g.t_count, g.eps2, static_cast<float4 *>(acc_dev), g.stream);
}

int colatus_trace(const int32_t *idx_dev, int k, void *ring_dev, int capacity_steps) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    if (k < 0) return fail(COLATUS_INVALID_ARG, "k < 0");
    invalidate_graph();
    if (k == 0) {
        g.trace_k = 0;
        return COLATUS_OK;
    }
    if (!idx_dev || !ring_dev || !aligned16(ring_dev)) return fail(COLATUS_INVALID_ARG, "null or misaligned pointer");
    if (capacity_steps < 1) return fail(COLATUS_INVALID_ARG, "capacity_steps < 1");
    g.trace_k = k;
    g.trace_cap = capacity_steps;
    g.ring = static_cast<float4 *>(ring_dev);
    int rc = build_trace_map(idx_dev);
    if (rc) g.trace_k = 0;
    return rc;
}

int colatus_trace_read(float *host_out, int64_t first_step, int n_steps) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded || g.trace_k == 0) return fail(COLATUS_NOT_UPLOADED, "no tracers configured");
    if (!host_out || n_steps < 1 || first_step < 0) return fail(COLATUS_INVALID_ARG, "bad arguments");
    if (first_step + n_steps > g.step || first_step < g.step - g.trace_cap)
        return fail(COLATUS_INVALID_ARG, "steps [%lld, +%d) not held by the ring (step=%lld, capacity=%d)",
                    (long long)first_step, n_steps, (long long)g.step, g.trace_cap);
    const size_t row = (size_t)g.trace_k * 16;
    for (int s = 0; s < n_steps;) {   // contiguous runs of ring rows
        const int64_t slot = (first_step + s) % g.trace_cap;
        int run = n_steps - s;
        if (slot + run > g.trace_cap) run = (int)(g.trace_cap - slot);
        CUDA_TRY(cudaMemcpyAsync(reinterpret_cast<unsigned char *>(host_out) + (size_t)s * row,
                                 reinterpret_cast<unsigned char *>(g.ring) + (size_t)slot * row, (size_t)run * row,
                                 cudaMemcpyDeviceToHost, g.stream));
        s += run;
    }
    CUDA_TRY(cudaStreamSynchronize(g.stream));
    return COLATUS_OK;
}

int colatus_splat(const void *pos_mass_dev, int64_t n, int axis, const float window[6], int width, int height,
                  uint32_t *image_dev, void *cuda_stream) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    const float4 *pm = static_cast<const float4 *>(pos_mass_dev);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (!pm) {
        if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "pos_mass_dev is null and colatus_upload has not been called");
        pm = g.pos;
        n = g.n;
        st = g.stream;
    }
    if (!window || !image_dev) return fail(COLATUS_INVALID_ARG, "null pointer");
    if (n < 1 || n > 2147483647LL) return fail(COLATUS_INVALID_ARG, "n=%lld out of [1, 2^31-1]", (long long)n);
    if (!aligned16(pm) || (reinterpret_cast<uintptr_t>(image_dev) & 3u))
        return fail(COLATUS_INVALID_ARG, "pointer misaligned");
    if (axis < 0 || axis > 2) return fail(COLATUS_INVALID_ARG, "axis must be 0, 1 or 2");
    if (width < 1 || width > 32768 || height < 1 || height > 32768)
        return fail(COLATUS_INVALID_ARG, "width and height must be in [1, 32768]");
    const float u0 = window[0], u1 = window[1], v0 = window[2], v1 = window[3], w0 = window[4], w1 = window[5];
    if (!std::isfinite(u0) || !std::isfinite(u1) || !std::isfinite(v0) || !std::isfinite(v1) || !(u1 > u0) ||
        !(v1 > v0) || !(w1 > w0))
        return fail(COLATUS_INVALID_ARG, "window needs finite u0 < u1, v0 < v1 and w0 < w1");
    const float su = (float)width / (u1 - u0);            // one IEEE single division each (reading G23)
    const float sv = (float)height / (v1 - v0);
    if (!std::isfinite(su) || !std::isfinite(sv)) return fail(COLATUS_INVALID_ARG, "window too narrow");
    CUDA_TRY(cudaMemsetAsync(image_dev, 0, (size_t)width * height * sizeof(uint32_t), st));
    splat_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(pm, n, axis, u0, su, v0, sv, w0, w1, width, height,
                                                              image_dev);
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    return COLATUS_OK;
}

int colatus_trace_spectrum(int64_t first_step, int n_steps, double *spectrum_dev) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded || g.trace_k == 0) return fail(COLATUS_NOT_UPLOADED, "no tracers configured");
    if (!spectrum_dev || (reinterpret_cast<uintptr_t>(spectrum_dev) & 7u))
        return fail(COLATUS_INVALID_ARG, "spectrum_dev null or misaligned");
    if (n_steps < 2 || n_steps > 65536 || first_step < 0)
        return fail(COLATUS_INVALID_ARG, "need first_step >= 0 and 2 <= n_steps <= 65536");
    if (first_step + n_steps > g.step || first_step < g.step - g.trace_cap)
        return fail(COLATUS_INVALID_ARG, "steps [%lld, +%d) not held by the ring (step=%lld, capacity=%d)",
                    (long long)first_step, n_steps, (long long)g.step, g.trace_cap);
    const int nf = n_steps / 2 + 1;
    const int bx = g.trace_k >= 32 ? 32 : (g.trace_k >= 16 ? 16 : 8);   // tracers across lanes
    const dim3 block(bx, 256 / bx);
    const dim3 grid((g.trace_k + block.x - 1) / block.x, (nf + block.y - 1) / block.y);
    trace_spectrum_kernel<<<grid, block, 0, g.stream>>>(g.ring, g.trace_k, g.trace_cap, first_step, n_steps,
                                                        spectrum_dev);
    CUDA_TRY(cudaGetLastError());
    g.launches++;
    return COLATUS_OK;
}

int colatus_diagnostics(double a, int with_potential, double out[16]) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    if (!out) return fail(COLATUS_INVALID_ARG, "out is null");
    if (!std::isfinite(a) || !(a > 0.0)) return fail(COLATUS_INVALID_ARG, "a must be finite and > 0");
    const Workspace w = workspace_layout(g.n);
    float4 *scratch = reinterpret_cast<float4 *>(g.ws + w.scratch_acc);
    double *partial = reinterpret_cast<double *>(g.ws + w.diag);
    if (with_potential) {
        int rc = run_forces(g.pos, g.n, g.t_begin, g.t_count, g.eps2, scratch, true, g.stream);
        if (rc) return rc;
    }
    int blocks = (int)((g.t_count + 255) / 256);
    if (blocks > DIAG_BLOCKS_MAX) blocks = DIAG_BLOCKS_MAX;
    diagnostics_partial_kernel<<<blocks, 256, 0, g.stream>>>(g.pos + g.t_begin, g.vel + g.t_begin,
                                                             with_potential ? scratch : nullptr, g.t_count, partial);
    CUDA_TRY(cudaGetLastError());
    double *final_dev = partial + (size_t)DIAG_BLOCKS_MAX * DIAG_Q;
    diagnostics_final_kernel<<<1, DIAG_Q * 32, 0, g.stream>>>(partial, blocks, final_dev);
    CUDA_TRY(cudaGetLastError());
    g.launches += 2;
    double q[DIAG_Q];
    CUDA_TRY(cudaMemcpyAsync(q, final_dev, sizeof(q), cudaMemcpyDeviceToHost, g.stream));
    CUDA_TRY(cudaStreamSynchronize(g.stream));
    out[0] = q[0];
    for (int c = 0; c < 3; ++c) {
        out[1 + c] = q[1 + c];
        out[4 + c] = a * a * q[1 + c];
        out[9 + c] = q[5 + c] / q[0];
    }
    out[7] = 0.5 * a * a * q[4];
    out[8] = with_potential ? 0.5 * q[8] / a : std::numeric_limits<double>::quiet_NaN();
    out[12] = (double)g.step;
    for (int c = 0; c < 3; ++c) out[13 + c] = q[5 + c];
    return COLATUS_OK;
}

int colatus_download(float *pos_mass_host, float *vel_host) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!g.uploaded) return fail(COLATUS_NOT_UPLOADED, "colatus_upload has not been called");
    if (pos_mass_host)
        CUDA_TRY(cudaMemcpyAsync(pos_mass_host, g.pos, (size_t)g.n * 16, cudaMemcpyDeviceToHost, g.stream));
    if (vel_host) CUDA_TRY(cudaMemcpyAsync(vel_host, g.vel, (size_t)g.n * 16, cudaMemcpyDeviceToHost, g.stream));
    CUDA_TRY(cudaStreamSynchronize(g.stream));
    return COLATUS_OK;
}

int colatus_profile(int enable) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    g.profile = enable != 0;
    g.ev_used = 0;
    return COLATUS_OK;
}

int colatus_profile_read(double *total_ms, int64_t *launches) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!total_ms || !launches) return fail(COLATUS_INVALID_ARG, "null pointer");
    double sum = 0.0;
    for (size_t i = 0; i + 1 < g.ev_used; i += 2) {
        CUDA_TRY(cudaEventSynchronize(g.ev_pool[i + 1]));
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, g.ev_pool[i], g.ev_pool[i + 1]));
        sum += ms;
    }
    *total_ms = sum;
    *launches = (int64_t)(g.ev_used / 2);
    g.ev_used = 0;
    return COLATUS_OK;
}

int64_t colatus_launch_count(void) { return g.launches; }

int colatus_force_geometry(int64_t n, int64_t target_count, int64_t out[8]) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!out || n < 1 || target_count < 1 || target_count > n) return fail(COLATUS_INVALID_ARG, "bad arguments");
    const Geometry geo = choose_geometry(n, target_count);
    out[0] = (int64_t)FORCE_THREADS * 2 * geo.IP;
    out[1] = geo.tiles_t;
    out[2] = geo.splits;
    out[3] = geo.sym ? geo.n_pad : (int64_t)geo.tiles_per_split * geo.TJ;
    out[4] = geo.sym && geo.IP > 3 ? 1 : g.ctas_per_sm;
    out[5] = g.sm_count;
    out[6] = 2 * geo.IP;
    out[7] = FORCE_THREADS;
    return COLATUS_OK;
}

int colatus_force_plan(int64_t n, int64_t target_count, int with_potential, int64_t out[8]) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!out || n < 1 || target_count < 1 || target_count > n) return fail(COLATUS_INVALID_ARG, "bad arguments");
    const Geometry geo = choose_geometry(n, target_count, with_potential != 0);
    out[0] = geo.sym ? 1 : 0;
    out[1] = geo.sym ? geo.nb : 0;
    out[2] = geo.splits;
    out[3] = geo.sym ? geo.H : 0;
    out[4] = geo.sym ? geo.K : 0;
    out[5] = geo.sym ? geo.chunks : 1;
    out[6] = geo.n_pad;
    out[7] = geo.sym ? geo.splits + (geo.H < geo.K ? geo.H : geo.K) : (geo.splits > 1 ? geo.splits : 0);
    return COLATUS_OK;
}

int colatus_set_option(const char *name, int64_t value) {
    if (!g.initialised) return fail(COLATUS_NOT_INITIALISED, "colatus_init has not been called");
    if (!name) return fail(COLATUS_INVALID_ARG, "name is null");
    if (!strcmp(name, "targets_per_thread")) {
        if (value != 0 && value != 2 && value != 4 && value != 6) return fail(COLATUS_INVALID_ARG, "must be 0,2,4,6");
        g.force_I = (int)value;
    } else if (!strcmp(name, "source_splits")) {
        if (value < 0 || value > MAX_SPLITS) return fail(COLATUS_INVALID_ARG, "must be in [0, %d]", MAX_SPLITS);   // capped per n
        g.force_splits = (int)value;
    } else if (!strcmp(name, "symmetric")) {
        if (value < 0 || value > 2) return fail(COLATUS_INVALID_ARG, "must be 0 (never), 1 (automatic) or 2 (always)");
        g.symmetric = (int)value;
    } else if (!strcmp(name, "symmetric_block")) {
        if (value != 0 && value != 1024 && value != 1536 && value != 4096)
            return fail(COLATUS_INVALID_ARG, "must be 0, 1024, 1536 or 4096");
        g.sym_block = (int)value;
    } else if (!strcmp(name, "symmetric_rows")) {
        if (value < 0 || value == 1 || value > 1000000) return fail(COLATUS_INVALID_ARG, "must be 0 or >= 2");
        g.sym_rows = (int)value;
    } else {
        return fail(COLATUS_INVALID_ARG, "unknown option %s", name);
    }
    invalidate_graph();
    return COLATUS_OK;
}

const char *colatus_last_error(void) { return g.err; }

}  // extern "C"

// ================================================================================================
// colatus_forces_static: eq. (1), for callers who have no device memory to give as a workspace.
//
// Every other entry point takes its scratch (staged sources, source-split partial sums, the equal-mass flag) from the
// workspace handed to colatus_init, which somebody had to cudaMalloc.  Some callers cannot: a plug-in running inside a
// host application whose own pool already owns the device memory, a callback or a tight control loop where a
// cudaMalloc (it synchronises the whole device and may fail late) is not acceptable, a process started with a fixed
// device-memory budget.  For them the same three kernels run here with their scratch in the file-scope device array
// below.  The array is part of the library's image: every GPU on which this library's module gets loaded sets
// COLATUS_STATIC_BYTES (4.5 MiB) aside until the process exits, used or not -- which is why the limit is modest.
//
// `static_scratch` is a device symbol.  In HOST code the name stands for a host-side shadow of it, not for a device
// address: a kernel handed `static_scratch` (or &static_scratch[0]) from host code would fault or, on a system whose
// GPU can reach host memory, quietly work on the wrong memory.  The device address is asked for once per device,
// with that device current, through cudaGetSymbolAddress, in this file (the symbol has file scope), and that pointer
// is what the kernels get.
namespace {

constexpr int64_t STATIC_MAX_N = COLATUS_STATIC_MAX_N;
constexpr int STATIC_TJ = 128;                        // force_kernel<1, 128, ...>: 512 targets per CTA, 128-source tiles
constexpr int STATIC_MAX_SPLITS = 16;                 // as the automatic choice of the workspace path: FP32 row sums
constexpr size_t STATIC_FLAG_BYTES = 256;
constexpr size_t STATIC_STAGED_BYTES = (size_t)(STATIC_MAX_N + STATIC_MAX_SPLITS * STATIC_TJ) * 16;
constexpr size_t STATIC_PARTIAL_CELLS = (size_t)8 * STATIC_MAX_N;   // float4 cells of partial sums: splits * n <= this
constexpr size_t COLATUS_STATIC_BYTES = STATIC_FLAG_BYTES + STATIC_STAGED_BYTES + STATIC_PARTIAL_CELLS * 16;
constexpr int STATIC_MAX_DEVICES = 64;

static __device__ __align__(256) unsigned char static_scratch[COLATUS_STATIC_BYTES];

struct StaticDevice {
    bool ready = false;
    unsigned char *base = nullptr;   // device address of static_scratch on this device
    int sm_count = 0;
};
StaticDevice static_dev[STATIC_MAX_DEVICES];

// Once per device, with that device current: the device address of the scratch array and the SM count.
int static_setup(int device, StaticDevice **out) {
    if (device < 0 || device >= STATIC_MAX_DEVICES)
        return fail(COLATUS_INVALID_ARG, "colatus_forces_static: device ordinal %d outside [0, %d)", device,
                    STATIC_MAX_DEVICES);
    StaticDevice &d = static_dev[device];
    if (!d.ready) {
        int major = 0, sms = 0;
        CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device));
        if (major != 10)
            return fail(COLATUS_UNSUPPORTED_DEVICE, "device %d is cc %d.x; libcolatus is built for sm_100a only", device,
                        major);
        CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
        void *p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&p, static_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u))
            return fail(COLATUS_CUDA_ERROR, "colatus_forces_static: scratch symbol resolved to %p", p);
        d.base = static_cast<unsigned char *>(p);
        d.sm_count = sms;
        d.ready = true;
    }
    *out = &d;
    return COLATUS_OK;
}

}  // namespace

extern "C" int colatus_forces_static(const void *pos_mass_dev, int64_t n, float eps2, double G, void *acc_out_dev,
                                     void *cuda_stream) {
    if (!pos_mass_dev || !acc_out_dev) return fail(COLATUS_INVALID_ARG, "null pointer");
    if (n < 1) return fail(COLATUS_INVALID_ARG, "n=%lld is below 1", (long long)n);
    if (n > STATIC_MAX_N)
        return fail(COLATUS_INVALID_ARG,
                    "colatus_forces_static: n=%lld exceeds COLATUS_STATIC_MAX_N=%lld, the size its built-in scratch "
                    "array is laid out for; larger problems need colatus_init with a workspace and colatus_forces",
                    (long long)n, (long long)STATIC_MAX_N);
    if (!aligned16(pos_mass_dev) || !aligned16(acc_out_dev)) return fail(COLATUS_INVALID_ARG, "pointer not 16-byte aligned");
    if (pos_mass_dev == acc_out_dev) return fail(COLATUS_INVALID_ARG, "pos_mass and acc_out alias");
    if (!eps2_ok(eps2)) return fail(COLATUS_INVALID_ARG, "eps2 must be finite and >= 1e-24");
    if (!std::isfinite(G)) return fail(COLATUS_INVALID_ARG, "G is not finite");
    int device = -1;
    CUDA_TRY(cudaGetDevice(&device));
    StaticDevice *d = nullptr;
    if (int rc = static_setup(device, &d)) return rc;

    // geometry: a pure function of (n, SM count), so the summation order -- and the bits -- repeat from call to call.
    // Enough source splits for two CTAs per SM, bounded by the partial-sum cells the array holds.
    const int64_t tiles_t = (n + 2 * FORCE_THREADS - 1) / (2 * FORCE_THREADS);
    const int64_t src_tiles = (n + STATIC_TJ - 1) / STATIC_TJ;
    int64_t splits = (2 * (int64_t)d->sm_count + tiles_t - 1) / tiles_t;
    if (splits > STATIC_MAX_SPLITS) splits = STATIC_MAX_SPLITS;
    if (splits > src_tiles) splits = src_tiles;
    if (splits > (int64_t)(STATIC_PARTIAL_CELLS / (size_t)n)) splits = (int64_t)(STATIC_PARTIAL_CELLS / (size_t)n);
    const int64_t tiles_per_split = (src_tiles + splits - 1) / splits;
    const int64_t n_pad = splits * tiles_per_split * STATIC_TJ;
    if ((size_t)n_pad * 16 > STATIC_STAGED_BYTES || (size_t)splits * (size_t)n > STATIC_PARTIAL_CELLS)
        return fail(COLATUS_INVALID_ARG, "colatus_forces_static: internal layout overflow at n=%lld", (long long)n);

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int *mass_flag = reinterpret_cast<int *>(d->base);
    float4 *staged = reinterpret_cast<float4 *>(d->base + STATIC_FLAG_BYTES);
    float4 *partials = reinterpret_cast<float4 *>(d->base + STATIC_FLAG_BYTES + STATIC_STAGED_BYTES);
    const float4 *pos_mass = static_cast<const float4 *>(pos_mass_dev);
    float4 *out = static_cast<float4 *>(acc_out_dev);

    // The array still holds what the previous call left.  Only the equal-mass flag has to start from zero (the staging
    // kernel stamps it when some mass differs from body 0's); the staged sources and every partial-sum cell the
    // reduction reads are written anew by this call's kernels.
    constexpr int generation = 1;
    CUDA_TRY(cudaMemsetAsync(mass_flag, 0, sizeof(int), st));
    stage_sources_kernel<<<(unsigned)((n_pad + 255) / 256), 256, 0, st>>>(pos_mass, n, n_pad, staged, mass_flag, generation);
    CUDA_TRY(cudaGetLastError());
    const bool single = splits == 1;
    CUDA_TRY(launch_ex(force_kernel<1, STATIC_TJ, NSTAGES, false, 2>, dim3((unsigned)tiles_t, (unsigned)splits),
                       dim3(FORCE_THREADS), force_smem_bytes<1, STATIC_TJ, NSTAGES, false>(), st, false, pos_mass,
                       (const float4 *)staged, (int64_t)0, n, (int)tiles_per_split, eps2, single ? (float)G : 1.0f,
                       single ? 1 : 0, single ? out : partials, n, (const int *)mass_flag, generation, (int *)nullptr));
    g.launches += 2;
    if (!single) {
        reduce_partials_kernel<false><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(partials, n, (int)splits, n, (float)G,
                                                                                  eps2, pos_mass, 0, out);
        CUDA_TRY(cudaGetLastError());
        g.launches++;
    }
    return COLATUS_OK;
}
