/*
 * colatus.h -- C ABI of libcolatus: the B200 (sm_100a) hot path of COLATUS,
 * arXiv 1208.3444 ("PAPER.md" below = /root/reference/PAPER.md).
 *
 * What the library computes
 *   - eq. (1), PAPER.md:29 : softened direct-summation acceleration
 *         F_k = G * sum_{j != k} m_j (x_j - x_k) / (|x_j - x_k|^2 + eps^2)^{3/2}
 *     (attractive sign, reading G1; the a^-3 of eq. (1) is applied in
 *     the kick, reading G5).  FP32 arithmetic, blocked FP32 accumulation.
 *   - eqs. (3)-(5), PAPER.md:38-44 : comoving drift-kick-drift leapfrog with the
 *     Hubble-drag factor (1-H tau)/(1+H tau); kick and second half-drift fused.
 *   - eq. (2), PAPER.md:33 : Friedmann equation, host only, double precision.
 *   - per-step velocities of selected tracer particles.
 *   - momentum / energy reductions (p = m a^2 v, eq. (7)).
 *   - a headless particle-count snapshot (Fig. 1) and the power spectrum of
 *     the tracer velocity series.
 *
 * Conventions
 *   - "body array" = float4 per particle, 16-byte aligned: positions carry
 *     (x, y, z, m) -- mass in .w as in the paper's kernel, PAPER.md:142 --
 *     velocities (vx, vy, vz, unused) and accelerations (ax, ay, az, w).
 *   - `*_dev` pointers are DEVICE pointers owned by the caller; `*_host`
 *     pointers are host pointers owned by the caller.  The library never
 *     allocates or frees device memory: scratch comes from the caller's
 *     workspace (colatus_workspace_bytes) -- or, for colatus_forces_static alone, from an
 *     array built into the library.  It keeps raw pointers only between
 *     colatus_upload / colatus_trace and colatus_shutdown.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).
 *   - One implicit process-wide context (one GPU per process).  Calls are not
 *     thread-safe; serialise them.
 *   - ONE workspace serves every entry point (staged sources, partial sums, the equal-mass flag,
 *     host-buffer staging, step table): work enqueued through this library must be stream-ordered
 *     as a whole.  Serialising the host calls is not enough -- two evaluations on different
 *     streams, or a colatus_forces* / colatus_splat call on a stream other than the resident one
 *     while resident work (colatus_step, colatus_run, colatus_diagnostics) is still in flight, race
 *     on the device.  Use one stream, or order the streams with events before each call.
 *   - Every function returning int returns COLATUS_OK (0) or a negative
 *     colatus_status; on error no output is written and colatus_last_error()
 *     describes the failure.  No exception or abort crosses the ABI.
 *   - There is no CPU fallback: without an sm_100 device colatus_init returns
 *     COLATUS_UNSUPPORTED_DEVICE or COLATUS_CUDA_ERROR.
 *   - Device data are not scanned: NaN/Inf inputs give NaN outputs, not errors.
 *   - Results of every call of this library are bit-reproducible run to run for a fixed
 *     (n, device, build, options): no floating-point atomics anywhere, all sums in a fixed order.
 *     That is a statement about ONE GPU.  Across GPUs (paper_1208_3444_b200/sharded.py) it carries
 *     over to target sharding, whose only exchange is an all-gather of positions (bits are moved,
 *     not added); in symmetric sharding the shares of colatus_forces_symmetric_part are summed by
 *     an FP32 all-reduce whose order belongs to the communication library, so forces there are
 *     reproducible only up to that summation order (never run on more than one GPU so far).
 *   - Equal masses are detected on the device at every force evaluation (all m_j equal to
 *     m_0 in value): the kernel then applies the common mass once to the finished sums instead
 *     of once per pair (one rounding fewer per term).  No flag, no host round trip; a NaN or a
 *     single different mass selects the general loop.  Positions must stay well below 1e18 in
 *     magnitude (padding bodies of mass 0 sit there).
 */
#ifndef COLATUS_H
#define COLATUS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum colatus_status {
    COLATUS_OK = 0,
    COLATUS_INVALID_ARG = -1,          /* null / misaligned pointer, n out of range, non-finite scalar ... */
    COLATUS_NOT_INITIALISED = -2,
    COLATUS_ALREADY_INITIALISED = -3,
    COLATUS_WORKSPACE_TOO_SMALL = -4,
    COLATUS_NOT_UPLOADED = -5,
    COLATUS_UNSUPPORTED_DEVICE = -6,   /* device is not compute capability 10.x */
    COLATUS_CUDA_ERROR = -7            /* text in colatus_last_error() */
} colatus_status;

/* colatus_config.flags */
#define COLATUS_FLAG_NONE 0u

typedef struct colatus_config {
    double   G;                 /* gravitational constant of eq. (1); finite */
    int      device;            /* CUDA device ordinal */
    void    *workspace_dev;     /* device scratch, 256-byte aligned, caller-owned */
    size_t   workspace_bytes;   /* >= colatus_workspace_bytes(n_max) for the largest n used */
    unsigned flags;             /* COLATUS_FLAG_* */
} colatus_config;

/* Cosmological model of eq. (2): H0 and the four density parameters today. */
typedef struct colatus_cosmo { double H0, Om_R, Om_M, Om_K, Om_L; } colatus_cosmo;

/* Bytes of device workspace needed for problems up to n_max bodies: the staged (padded)
 * source array, the partial-sum rows, reduction scratch, and staging for the host-buffer
 * entry point.  From 20480 bodies on the partial rows are those of the symmetric force kernel
 * (colatus_force_plan): one row of 16 bytes per body for every source split and every block
 * distance while that fits 512 MiB, else 32 rows, the evaluation then taking several launches
 * (measured cost of the smaller budget: +0.7 % at 2^20, +0.4 % at 2^22).  About 1.1 to 1.4 KB per
 * body up to 65536 bodies (5.5 MiB at n = 4096, 37 MiB at 32768), 91 MiB at 131072, 0.55 GiB at
 * 524288, 0.59 GiB at 2^20, 2.36 GiB at 2^22, 9.4 GiB at 2^24 (0.6 KB per body from 2^20 on).
 * The size depends on n_max alone (not on the device or on options).  Non-decreasing in n_max: a
 * workspace sized for n_max serves every n <= n_max.  Pure host arithmetic; 0 if n_max < 1. */
size_t colatus_workspace_bytes(int64_t n_max);

/* Selects the device, checks it is cc 10.x, records G and the workspace.  A second
 * call without colatus_shutdown returns COLATUS_ALREADY_INITIALISED. */
int  colatus_init(const colatus_config *cfg);
void colatus_shutdown(void);

/* ---- eq. (1): stateless force evaluation on caller-owned device arrays -------------
 * pos_mass_dev : const float4[n]  (x, y, z, m)
 * acc_out_dev  : float4[n]        (F_x, F_y, F_z, 0)  with G applied, a^-3 NOT applied
 * eps2         : eps^2 (the paper's min_dist^2), finite, >= 1e-24.  The j = k term is not
 *                branched around (reading G4): it is m_k eps2^-1.5 * 0 = 0 exactly, PROVIDED m_k eps2^-1.5 is
 *                finite in FP32 -- the caller keeps |m| * eps2^-1.5 < 3e38 (at the floor: |m| < 3e2), else
 *                that target's force is NaN.  The same bound keeps close distinct pairs finite.
 * Whole-range evaluations of >= 20480 bodies evaluate every pair once and apply it to both bodies
 * (the symmetric kernel, colatus_force_plan); results agree with the one-directional kernel to FP32
 * summation rounding, and either is bitwise reproducible from run to run.
 * Enqueues on cuda_stream and returns without synchronising.  n in [1, 2^31-1];
 * pointers 16-byte aligned and distinct. */
int colatus_forces(const void *pos_mass_dev, int64_t n, float eps2, void *acc_out_dev,
                   void *cuda_stream);

/* As colatus_forces but acc_out[k].w = phi_k = -G sum_{j != k} m_j / sqrt(r^2 + eps^2)
 * (the potential whose gradient is eq. (1); used for the energy of eq. (7)). */
int colatus_forces_potential(const void *pos_mass_dev, int64_t n, float eps2, void *acc_out_dev,
                             void *cuda_stream);

/* Forces on targets [target_begin, target_begin + target_count) only, all n bodies acting
 * as sources; acc_out_dev is float4[target_count].  The multi-GPU path shards eq. (1) by
 * targets with this call. */
int colatus_forces_range(const void *pos_mass_dev, int64_t n, int64_t target_begin,
                         int64_t target_count, float eps2, void *acc_out_dev, void *cuda_stream);

/* One share of a SYMMETRIC evaluation of eq. (1) (colatus_force_plan): the block pairs whose target
 * block lies in share `part` of `parts` -- contiguous ranges of the blocks, equal work because the pairing is
 * circulant.  acc_out_dev = float4[n], ALL bodies: G x what those pairs deliver, to their own blocks and, as
 * reactions (Newton's third law), to the blocks they meet; exactly 0 for bodies they do not reach.  The outputs of
 * the shares 0 .. parts-1 add up to the whole force: this is how eq. (1) is divided over GPUs without giving up the
 * single evaluation of every pair -- every GPU holds all positions (one all-gather per step, as for target sharding),
 * evaluates share `rank` of `world`, and ONE all-reduce of the float4[n] outputs gives every GPU the forces
 * (paper_1208_3444_b200/sharded.py).  Any n for which the workspace holds two partial rows (else INVALID_ARG).
 * The eq. (10) source and the background term are NOT part of a share (they would be counted `parts` times): a
 * driver adds them once to the summed forces with colatus_add_external.
 * Same argument rules as colatus_forces; enqueues on cuda_stream. */
int colatus_forces_symmetric_part(const void *pos_mass_dev, int64_t n, float eps2, int part, int parts,
                                  void *acc_out_dev, void *cuda_stream);

/* Host-buffer variant: copies float4[n] host -> device, evaluates eq. (1), copies
 * float4[n] back and synchronises.  Uses the workspace staging area and the stream given
 * (NULL = default).  This is the end-to-end call bench.py's "e2e" times. */
int colatus_forces_host(const float *pos_mass_host, int64_t n, float eps2, float *acc_out_host,
                        void *cuda_stream);

/* ---- eq. (1), for callers who cannot allocate device memory ----------------
 * colatus_forces needs a workspace, and a workspace is something somebody cudaMalloc'ed.  Not every caller can do
 * that: code running inside an application whose own memory pool already owns the device memory, a callback or
 * control loop that must not hit cudaMalloc's device-wide synchronisation (or its late out-of-memory failure), a
 * process held to a fixed device-memory budget.  This ONE entry point serves them: it needs neither colatus_init
 * nor a workspace, and it calls no cudaMalloc, cudaFree or any other allocating routine.  Its scratch (staged
 * sources, source-split partial sums, the equal-mass flag) is an array built into the library's device image --
 * about 4.5 MiB, which every GPU that loads this library's kernels holds until the process exits, whether or not
 * this function is ever called.  That is the reason for the modest limit:
 *     1 <= n <= COLATUS_STATIC_MAX_N  (32768 = 32^3, the largest run of the paper);
 * larger n is refused with COLATUS_INVALID_ARG and a message naming the limit (use colatus_forces then).
 * pos_mass_dev : const float4[n] (x, y, z, m), acc_out_dev : float4[n] (F_x, F_y, F_z, 0) -- device memory the
 * caller already owns, 16-byte aligned, distinct; eps2 as for colatus_forces; G = the constant of eq. (1), finite
 * (there is no context to take it from).  Same kernels and arithmetic as colatus_forces' one-directional path with
 * a fixed geometry (2 targets per thread, up to 16 source splits -- a pure function of n and the SM count), so
 * results agree with colatus_forces to FP32 summation rounding and repeat bit for bit from call to call.  The
 * eq. (10) source and the background term of colatus_set_deformation / _background are NOT added.
 * Runs on the CURRENT device (cudaGetDevice); enqueues on cuda_stream and returns without synchronising.
 * The first call on each device also does a one-time set-up (looks up the array's device address and the SM
 * count, which may make the driver load the library's device code): make that first call outside any stream
 * capture.  All calls share the one array, and it keeps what the last call left -- the function clears the
 * one word that has to start at zero itself -- so two calls whose work overlaps on the GPU (different streams,
 * no ordering between them) race; order them on one stream or with events.  Independent of the workspace: it
 * may be mixed freely with the other entry points.  Not thread-safe, like the rest of the library. */
#define COLATUS_STATIC_MAX_N 32768
int colatus_forces_static(const void *pos_mass_dev, int64_t n, float eps2, double G, void *acc_out_dev,
                          void *cuda_stream);

/* ---- eqs. (3)-(5): resident simulation state ----------------------------------------
 * Binds caller-owned device buffers (float4[n] each); all later step work is enqueued
 * on `cuda_stream`.  Resets the step counter to 0.  acc_dev receives F(x^{n+1/2}) of
 * the latest step. */
int colatus_upload(void *pos_mass_dev, void *vel_dev, void *acc_dev, int64_t n, float eps2,
                   void *cuda_stream);

/* One step of eqs. (3)-(5) with constant tau:
 *   x += tau/2 v;  F = eq.(1)(x);  v = v (1-H tau)/(1+H tau) + F tau/(a^3 (1+H tau));  x += tau/2 v
 * a, H are the caller's mid-step values (reading G3); the coefficients are formed in
 * double on the host and passed to the kernels as float.  Requires finite arguments,
 * a > 0 and 1 + H tau > 0.  Asynchronous. */
int colatus_step(double tau, double a, double H);

/* The four coefficients colatus_step uses, formed in double from eqs. (3)-(5):
 * out = { d1 = tau/2, cv = (1-H tau)/(1+H tau), ck = tau/(a^3 (1+H tau)), d2 = tau/2 }.
 * Host only; same argument checks as colatus_step. */
int colatus_step_coefficients(double tau, double a, double H, double out[4]);

/* Generic drift-kick-drift:  x += d1 v;  F = eq.(1)(x);  v = cv v + ck F;  x += d2 v.
 * Covers the symplectic operators of eq. (9), with v standing for p/m.
 * Asynchronous. */
int colatus_step_coeffs(double d1, double cv, double ck, double d2);

/* ---- native step loop ("optionally replayed from a CUDA graph") -----------------------
 * n_steps steps of eqs. (3)-(5) in one call, with the scale-factor schedule of eq. (2) formed
 * on the host in double exactly as a caller of colatus_step would: for each step
 *   a_mid = a(t_n + tau/2), H_mid = H(a_mid)  (reading G3),  then a(t_n + tau);
 * c == NULL means a static background (a = 1, H = 0; a_start ignored).  The per-step
 * coefficients go to a device table (in the workspace, 1024 steps per upload) and a device
 * counter selects the row, so every step launches the same kernels with the same arguments.
 * Whole-range runs without external terms take TWO launches per step: the force kernel, and one
 * tail/head kernel (partial-sum reduction + kick + drift + tracer record of step s, then the first
 * half drift + source staging of step s+1 -- two separately rounded drifts, as in colatus_step),
 * chained by programmatic dependent launch; only the first head of a run is a launch of its own.
 * With use_graph != 0 captured CUDA graphs of 8 steps (and of 1 step for the remainder) are
 * replayed -- this is what makes the launch-bound small-N loops (configs 1-3) fast; with
 * use_graph == 0 the same kernels are launched one by one.  Target sub-ranges and runs with
 * external terms take drift / force (+ reduction, external terms) / kick-drift launches instead.
 * Results are bitwise identical to n_steps calls of colatus_step.
 * The loop runs on a stream owned by the library, ordered after everything already enqueued
 * on the resident stream and before everything enqueued on it later.  *a_end (may be NULL)
 * receives a(t_0 + n_steps tau).  Nothing is enqueued if any step's coefficients are invalid
 * (colatus_step's checks).  The graph is re-captured after colatus_upload, colatus_trace,
 * colatus_set_target_range, colatus_set_deformation / _background or colatus_set_option.
 * Asynchronous. */
int colatus_run(const struct colatus_cosmo *c, double a_start, double tau, int64_t n_steps, int use_graph,
                double *a_end);
/* The same loop with the symplectic operators of eq. (9): per step the coefficients of
 * colatus_symplectic_coefficients (drift and kick integrals along eq. (2), FP64 on the host); the resident
 * "velocity" array holds w = a^2 v; tracer tag = a(t + tau).  c == NULL reduces to the static leapfrog.
 * Bitwise identical to n_steps calls of colatus_step_symplectic. */
int colatus_run_symplectic(const struct colatus_cosmo *c, double a_start, double tau, int64_t n_steps,
                           int use_graph, double *a_end);

/* ---- eq. (9): symplectic drift-kick-drift (reading G11) ---------------
 * The resident "velocity" array then holds w = p/m = a^2 v (canonical momentum per unit mass).
 *   D(tau/2): x += w * int_{t}^{t+tau/2} dt/a^2;   K(tau): w += F(x) * int_{t}^{t+tau} dt/a;
 *   D(tau/2): x += w * int_{t+tau/2}^{t+tau} dt/a^2
 * with F = eq. (1) (the comoving potential of eq. (1) plays the role of phi' in eq. (8): d(a^2 v)/dt = F/a).
 * colatus_symplectic_coefficients integrates eq. (2) from a(t) = a0 in double on the host and returns
 * out = { d1, cv = 1, ck, d2, a(t+tau) }; host only.  colatus_step_symplectic enqueues the step with those
 * coefficients (tracer tag = a(t+tau) as float) and returns a(t+tau) in *a_end (may be NULL).
 * Requires c != NULL, a0 > 0, finite tau.  Asynchronous. */
int colatus_symplectic_coefficients(const struct colatus_cosmo *c, double a0, double tau, double out[5]);
int colatus_step_symplectic(const struct colatus_cosmo *c, double a0, double tau, double *a_end);

/* ---- eq. (10): deformation-potential source (reading G21) -------------
 * A fixed point source at x_psi of strength S = C*psi that "acts like a mass particle located in a fixed
 * position": every force this library returns or uses gains
 *   F_k += S (x_psi - x_k) / (|x_k - x_psi|^2 + eps^2)^{3/2}
 * (attractive for S > 0; S is NOT multiplied by G, as in eq. (10)).  S = 0 disables (default).
 * The term is not part of acc.w / W.  Applies to colatus_forces, _potential, _range, _host, colatus_step*, colatus_run*
 * and colatus_force_kick_drift alike; the two calls that handle caller-assembled forces -- colatus_forces_symmetric_part
 * (a share) and colatus_kick_drift (forces as given) -- leave it to colatus_add_external, and colatus_forces_static
 * (no context) never adds it.  Host call. */
int colatus_set_deformation(const double x_psi[3], double strength);

/* Mean-density background term (reading G22; the paper states periodic/homogeneous
 * boundaries, but prints no algorithm): every force gains
 *   F_k += (4 pi / 3) G rho_bar (x_k - centre)
 * which cancels the net pull of a homogeneous sphere of comoving density rho_bar about `centre`, so
 * that an unperturbed box no longer contracts as a whole (G7).  rho_bar = 0 disables (default). */
int colatus_set_background(const double centre[3], double rho_bar);

/* Restrict the resident state to targets [target_begin, target_begin+target_count): only
 * those bodies are drifted, kicked and receive forces; all n bodies stay sources.  Used by
 * the target-sharded multi-GPU driver, which all-gathers positions between steps.
 * Default after colatus_upload is the full range. */
int colatus_set_target_range(int64_t target_begin, int64_t target_count);

/* Drift alone (eq. (3)): x += d v on the resident state's target range.  Asynchronous. */
int colatus_drift(double d);
/* Force on the resident state's target range into acc_dev, then the fused kick-drift
 * (eqs. (4)-(5)) v = cv v + ck F; x += d2 v and the tracer record.  Asynchronous. */
int colatus_force_kick_drift(double cv, double ck, double d2);
/* The kick-drift alone, with forces the caller supplies: acc_dev = const float4[target_count] (F of the target
 * range's bodies, G applied, indexed from the range's first body) -> v = cv v + ck F; x += d2 v, tracer record,
 * step counter + 1.  This is the second half of colatus_force_kick_drift for drivers that assemble F themselves
 * (the sharded symmetric evaluation: colatus_forces_symmetric_part on every GPU, one all-reduce).  Asynchronous. */
int colatus_kick_drift(const void *acc_dev, double cv, double ck, double d2);
/* The external terms for forces the caller assembled itself.  colatus_forces_symmetric_part returns SHARES of
 * eq. (1) that are summed over GPUs, so it cannot add the eq. (10) source or the
 * background term -- they would be counted once per share -- and colatus_kick_drift takes its forces as given.  This
 * call adds both terms, as set by colatus_set_deformation / colatus_set_background, ONCE to acc_dev = float4[target_count]
 * (forces of the resident target range's bodies, indexed from the range's first body) at the resident positions: the
 * sharded symmetric driver calls it between its all-reduce and colatus_kick_drift.  Nothing is launched when both terms
 * are off.  Do not apply it to the output of colatus_forces / _range (those already contain the terms).  Asynchronous
 * on the resident stream. */
int colatus_add_external(void *acc_dev);

/* ---- tracers -------------------------------------------------
 * After each step the velocities v^{n+1} of the k particles idx_dev[0..k) are written to
 * ring_dev[(step % capacity_steps)][k] as float4 (vx, vy, vz, tag) where tag is the
 * `trace_tag` of that step (colatus_step passes a as float; step_coeffs passes 0).
 * k = 0 disables tracing.  idx_dev: const int32[k]; ring_dev: float4[capacity_steps][k]. */
int colatus_trace(const int32_t *idx_dev, int k, void *ring_dev, int capacity_steps);

/* Copies steps [first_step, first_step+n_steps) of the ring to host_out[n_steps][k][4];
 * fails with COLATUS_INVALID_ARG if the ring no longer (or not yet) holds them.
 * Synchronises the stream. */
int colatus_trace_read(float *host_out, int64_t first_step, int n_steps);

/* ---- headless snapshot (NEXT row f4; App. A step 7, Fig. 1) ------
 * Particle-count image of the positions: the content of the paper's live display and of its
 * Fig. 1 panels, without a window (reading G23 -- the paper gives no rendering algorithm).
 * Orthographic projection along `axis` (0, 1, 2); image axes (u, v) = the two other
 * coordinates in cyclic order (axis 0: u=y, v=z; axis 1: u=z, v=x; axis 2: u=x, v=y); depth
 * w = coordinate `axis`.  window = (u0, u1, v0, v1, w0, w1) (host floats).  A body is counted
 * iff w0 <= w < w1 and 0 <= tu < width and 0 <= tv < height, where, in FP32 with each operation
 * rounded once, tu = (u - u0) * (width / (u1 - u0)), tv likewise; its pixel is
 * image_dev[floor(tv) * width + floor(tu)] (uint32, row-major [height][width], caller-owned
 * device memory, zeroed by this call).  Masses are ignored.  Counts are exact integers,
 * independent of execution order.
 * pos_mass_dev: device float4[n], or NULL for the resident state (then n is ignored and the
 * work goes to the resident stream).  Requirements: u1 > u0, v1 > v0, w1 > w0; u/v bounds
 * finite (w0, w1 may be -inf / +inf: no slab); 1 <= width, height <= 32768.  Asynchronous. */
int colatus_splat(const void *pos_mass_dev, int64_t n, int axis, const float window[6], int width,
                  int height, uint32_t *image_dev, void *cuda_stream);

/* ---- tracer velocity power spectrum (NEXT row f3) -------------------------------
 * "computation of the velocity of a single particle at every time-step ... and its energy
 * power spectrum": periodogram of the recorded series of every tracer (reading G24 -- the
 * paper gives no formula), summed over the velocity components:
 *   P_t[f] = (1/S) sum_c | sum_{s<S} v_{t,c}[first_step + s] exp(-2 pi i f s / S) |^2,
 *   f = 0 .. S/2,  S = n_steps,
 * so that the full-circle sum of P_t equals sum_s |v_t[s]|^2 (Parseval).
 * spectrum_dev: device double[k][S/2 + 1], caller-owned.  Direct O(k S^2) evaluation in FP64
 * from the FP32 ring samples.  The ring must still hold steps [first_step, first_step + S)
 * (as for colatus_trace_read); 2 <= S <= 65536.  Asynchronous on the resident stream. */
int colatus_trace_spectrum(int64_t first_step, int n_steps, double *spectrum_dev);

/* ---- diagnostics (eq. (7)) ------------------------------
 * Sums over the resident target range (all n bodies unless colatus_set_target_range):
 * out[0] = M = sum m;  out[1..3] = P = sum m v;  out[4..6] = a^2 P;
 * out[7] = T = 1/2 sum m a^2 v^2;  out[8] = W = -(G/2a) sum_k sum_{j!=k} m_k m_j/sqrt(r^2+eps^2)
 * with k over the range and j over all n (NaN unless with_potential, which costs a second
 * O(n^2) pass);  out[9..11] = sum m x / M;  out[12] = steps taken;  out[13..15] = sum m x
 * (so that shards can be added).  FP64 accumulation in a fixed order.  Synchronises the stream. */
int colatus_diagnostics(double a, int with_potential, double out[16]);

/* Copies the resident positions / velocities to host arrays float[n][4] (either may be
 * NULL).  Synchronises the stream. */
int colatus_download(float *pos_mass_host, float *vel_host);

/* ---- instrumentation ------------------------------------------------------------------
 * (Device microbenchmarks -- FP32 peak calibration, issue-rule probes -- are NOT here: they live in the
 * separate libcolatus_probe, include/colatus_probe.h.)
 * colatus_profile(1) makes the library bracket every force-kernel launch with CUDA events
 * on the launching stream; colatus_profile_read synchronises and returns the number of
 * bracketed launches and their summed duration in ms, then resets both.
 * colatus_launch_count returns the number of kernels this library has launched. */
int      colatus_profile(int enable);
int      colatus_profile_read(double *total_ms, int64_t *launches);
int64_t  colatus_launch_count(void);

/* Geometry the force path picked for n bodies / target_count targets on this device:
 * out[0] = targets per CTA, out[1] = target tiles, out[2] = source splits,
 * out[3] = sources per split (padded), out[4] = CTAs per SM, out[5] = SM count,
 * out[6] = kernel variant (targets per thread = 2 x target pairs), out[7] = threads per CTA. */
int colatus_force_geometry(int64_t n, int64_t target_count, int64_t out[8]);

/* Which force kernel an evaluation of target_count targets out of n bodies takes (eq. 1).
 * Whole-range evaluations (target_count == n) of at least 20480 bodies use the SYMMETRIC kernel: the pair term (x_j - x_k)/(r^2 + eps^2)^{3/2} is antisymmetric, so it is evaluated once
 * per unordered pair and applied to both bodies (Newton's third law) -- 16 packed FP32 operations per
 * 4 pair-interactions instead of 24.  Bodies are cut into blocks of 4096 (1024 below 65536 bodies); block a meets the `distances`
 * blocks a+1 .. a+distances (mod blocks) both ways, and itself (and the antipodal block when `blocks` is even)
 * one way.  The sums a block receives from each distance are kept as partial rows in the workspace and
 * added in fixed row order (in FP64 when there are more than 16 rows), so results are reproducible bit for
 * bit; when the rows of all distances exceed the workspace's row budget (512 MiB, or 32 rows if that is more:
 * from 2^20 bodies on) the evaluation runs as `launches` kernel launches of `distances_per_launch` distances each,
 * whose sums are carried in FP64 and rounded once.  Potential evaluations (with_potential != 0) carry the potential as a
 * fourth component through the same kernel, always with 1024-body blocks.  Target sub-ranges and smaller
 * problems take the one-directional kernel (out[0] = 0; its geometry is colatus_force_geometry's).
 * out[0] = 1 symmetric / 0 one-directional, out[1] = blocks, out[2] = splits of a block's work (CTAs = blocks x
 * splits), out[3] = distances H = (blocks-1)/2, out[4] = distances per launch, out[5] = launches,
 * out[6] = padded bodies, out[7] = partial rows added per body (0: none). */
int colatus_force_plan(int64_t n, int64_t target_count, int with_potential, int64_t out[8]);

/* Tuning overrides for measurements (0 restores the automatic choice):
 *   "targets_per_thread" in {0,2,4,6} (non-zero also selects the one-directional kernel);
 *   "source_splits" in [0,64] (capped at 16 above 65536 bodies; for the symmetric kernel at 32, 16 and 24 with
 *                blocks of 1024, 1536 and 4096 bodies);
 *   "symmetric": 0 = never use the symmetric kernel, 1 = automatic (default after colatus_init),
 *                2 = whenever the evaluation allows it (any n; for tests);
 *   "symmetric_block": bodies per block of the symmetric kernel, 1024, 1536 or 4096 (0 = automatic: 1024 below
 *                65536 bodies, 4096 from there on);
 *   "symmetric_rows": cap on the partial rows one launch of the symmetric kernel may use (0 = what the
 *                workspace holds, else >= 2): a small value splits an evaluation into several launches. */
int colatus_set_option(const char *name, int64_t value);

const char *colatus_last_error(void);

/* ---- host-only cosmology, FP64 (eq. (2)) ---------------------------------- */

/* H(a) = H0 sqrt(Om_R a^-4 + Om_M a^-3 + Om_K a^-2 + Om_L).  NaN if a <= 0. */
double colatus_hubble(const colatus_cosmo *c, double a);
/* a(t0 + dt) given a(t0) = a0, integrating da/dt = a H(a) (adaptive step doubling). */
double colatus_a_advance(const colatus_cosmo *c, double a0, double dt);
/* t(a) = integral_0^a da' / (a' H(a'));  +inf if it diverges (no matter, radiation or curvature). */
double colatus_time_of_a(const colatus_cosmo *c, double a);
/* integral_{t0}^{t0+dt} dt / a(t)^p with a(t0) = a0: drift (p=2) and kick (p=1) integrals of eq. (9). */
double colatus_int_dt_over_a_pow(const colatus_cosmo *c, double a0, double dt, double p);

#ifdef __cplusplus
}
#endif
#endif /* COLATUS_H */
