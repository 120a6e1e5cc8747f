/*
 * colatus_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what the COLATUS hot path
 * computes (arXiv 1208.3444), written from the paper so a reader can check it
 * against PAPER.md by eye.  It shares no code, header, table or helper with
 * the CUDA path under paper_1208_3444_b200/ and neither imports the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.
 *
 * Every function cites the passage it follows.  Readings of garbled or
 * ambiguous passages are the G-numbered ones in DESIGN.md ("Readings").
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"):
 *   oracle_forces      P1 closed-form two-body + exact rational three-body,
 *                      P2 third law, P3 softened-shell closed form,
 *                      P4 brute force tiny N, P5 symmetries, P6 monopole
 *   oracle_step        P8 static leapfrog (orbit, tau^2 energy error, time
 *                      reversal), P9 drag closed form + one-step worked example
 *   oracle_hubble / oracle_a_advance / oracle_time_of_a
 *                      P7 closed-form a(t) for EdS, flat LCDM, radiation,
 *                      matter+radiation, Milne, open matter+curvature, de Sitter
 *   oracle_diagnostics P9 momentum law, P11 Layzer-Irvine, static energy
 *   oracle_step_coeffs / oracle_int_dt_over_a_pow (symplectic step of eq. 9)
 *                      P12 EdS closed-form kick/drift integrals, exact sum m w
 *                      conservation, force-free closed form, agreement with
 *                      eqs. (3)-(5) as tau -> 0 at second order
 *   oracle_add_external P13 extra-body equivalence + two-body closed form (eq. 10),
 *                      linear closed form + homogeneous-sphere cancellation
 *   oracle_forces + oracle_step  P16 cold homogeneous sphere vs the scalar shell recurrence
 *   oracle_splat       P14 brute-force counts, total = in-window particles
 *   oracle_trace_spectrum P15 sinusoid closed form, Parseval, numpy FFT
 * Unpinned: nothing in this file.  (Physical realism of config 2 against the
 * paper's Fig. 1 statistics is "parity unpinned": it needs the paper's ICs.)
 *
 * Parallelism: OpenMP over targets only; the summation order inside one
 * target is fixed (j = 0..N-1), so results do not depend on the thread count.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * Eq. (1), with the attractive sign (reading G1) and WITHOUT the
 * a^-3 factor (reading G5: a^-3 belongs to eq. 4):
 *
 *   F_k = G * sum_{j != k} m_j (x_j - x_k) / (|x_j - x_k|^2 + eps^2)^{3/2}
 *
 * and the matching potential  phi_k = -G sum_{j != k} m_j / sqrt(|..|^2+eps^2)
 * (so that F_k = -grad_k phi).  Self term skipped by index as in the paper's
 * loop `if (idx != i)`, PAPER.md:138 (reading G4).
 *
 *   x        [n][3] positions (double)
 *   m        [n]    masses
 *   targets  [n_targets] indices k to evaluate, or NULL for k = 0..n_targets-1
 *   acc_out  [n_targets][3]
 *   phi_out  [n_targets] or NULL
 */
void oracle_forces(const double *x, const double *m, int64_t n, double eps2, double G,
                   const int64_t *targets, int64_t n_targets, double *acc_out, double *phi_out)
{
    int64_t t;
#pragma omp parallel for schedule(dynamic, 16)
    for (t = 0; t < n_targets; ++t) {
        const int64_t k = targets ? targets[t] : t;
        const double xk = x[3 * k + 0], yk = x[3 * k + 1], zk = x[3 * k + 2];
        double ax = 0.0, ay = 0.0, az = 0.0, phi = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == k) continue;
            const double dx = x[3 * j + 0] - xk;
            const double dy = x[3 * j + 1] - yk;
            const double dz = x[3 * j + 2] - zk;
            const double s = dx * dx + dy * dy + dz * dz + eps2;   /* r^2 + eps^2 */
            const double root = sqrt(s);
            const double w = m[j] / (s * root);                    /* m_j / (..)^{3/2} */
            ax += w * dx;
            ay += w * dy;
            az += w * dz;
            phi -= m[j] / root;
        }
        acc_out[3 * t + 0] = G * ax;
        acc_out[3 * t + 1] = G * ay;
        acc_out[3 * t + 2] = G * az;
        if (phi_out) phi_out[t] = G * phi;
    }
}

/*
 * One step of the difference equations (3)-(5), in the paper's
 * order: half drift, force at the half-step positions, kick with the Hubble
 * drag factor, half drift.  `a`, `H` are the values the caller evaluates at
 * the mid-step time (reading G3); `grad phi` in eq. (4) is read as the force F
 * of eq. (1) (reading G2).
 *
 *   x^{n+1/2} = x^n + (tau/2) v^n                                         (3)
 *   v^{n+1}   = v^n (1 - H tau)/(1 + H tau) + F(x^{n+1/2}) tau / (a^3 (1 + H tau))   (4)
 *   x^{n+1}   = x^{n+1/2} + (tau/2) v^{n+1}                               (5)
 *
 * x, v: [n][3] updated in place; m: [n]; work: [n][3] scratch for F.
 */
void oracle_step(double *x, double *v, const double *m, int64_t n, double eps2, double G,
                 double tau, double a, double H, double *work)
{
    int64_t i;
    for (i = 0; i < 3 * n; ++i) x[i] = x[i] + 0.5 * tau * v[i];                 /* (3) */
    oracle_forces(x, m, n, eps2, G, NULL, n, work, NULL);                        /* (1) */
    for (i = 0; i < 3 * n; ++i)                                                  /* (4) */
        v[i] = v[i] * (1.0 - H * tau) / (1.0 + H * tau)
             + work[i] * tau / (a * a * a * (1.0 + H * tau));
    for (i = 0; i < 3 * n; ++i) x[i] = x[i] + 0.5 * tau * v[i];                 /* (5) */
}

/*
 * Generic drift-kick-drift with caller-supplied coefficients
 *   x += d1 v;  F = F(x);  v = cv v + ck F;  x += d2 v
 * used for the symplectic variant of eq. (9), PAPER.md:64 (reading G11), where
 * d1, d2 = integral dt/a^2 over each half step and ck = integral dt/a, cv = 1,
 * with the variable w = p/m = a^2 v in place of v.
 */
void oracle_step_coeffs(double *x, double *v, const double *m, int64_t n, double eps2, double G,
                        double d1, double cv, double ck, double d2, double *work)
{
    int64_t i;
    for (i = 0; i < 3 * n; ++i) x[i] = x[i] + d1 * v[i];
    oracle_forces(x, m, n, eps2, G, NULL, n, work, NULL);
    for (i = 0; i < 3 * n; ++i) v[i] = cv * v[i] + ck * work[i];
    for (i = 0; i < 3 * n; ++i) x[i] = x[i] + d2 * v[i];
}

/*
 * External terms added to the force of eq. (1) (NEXT rows f2 and f5 of SURVEY 8f):
 *
 *  (a) eq. (10): the deformation-potential source, a fixed point at
 *      x_psi of strength S = C*psi which "acts like a mass particle located in a
 *      fixed position"; attractive sign as in reading G1, S not
 *      multiplied by G (reading G21):
 *          F_k += S (x_psi - x_k) / (|x_k - x_psi|^2 + eps^2)^{3/2}
 *  (b) mean-density background (reading G22; the paper asserts homogeneous /
 *      periodic boundaries, without an algorithm):
 *          F_k += (4 pi / 3) G rho_bar (x_k - centre)
 *
 * targets NULL = k = 0..n_targets-1.  acc [n_targets][3] is updated in place.
 * Pins: (a) equals oracle_forces with one more body of mass S/G at x_psi, and the
 * two-body closed form; (b) linear closed form, and cancellation of the pull of a
 * homogeneous sphere (tests/test_oracle_pins.py).
 */
void oracle_add_external(const double *x, const int64_t *targets, int64_t n_targets, double eps2,
                         double S, const double *x_psi, double G, double rho_bar, const double *centre,
                         double *acc)
{
    const double pi = 3.14159265358979323846;
    int64_t t;
    for (t = 0; t < n_targets; ++t) {
        const int64_t k = targets ? targets[t] : t;
        if (S != 0.0) {
            const double dx = x_psi[0] - x[3 * k], dy = x_psi[1] - x[3 * k + 1], dz = x_psi[2] - x[3 * k + 2];
            const double s = dx * dx + dy * dy + dz * dz + eps2;
            const double w = S / (s * sqrt(s));
            acc[3 * t] += w * dx;
            acc[3 * t + 1] += w * dy;
            acc[3 * t + 2] += w * dz;
        }
        if (rho_bar != 0.0) {
            const double B = (4.0 * pi / 3.0) * G * rho_bar;
            acc[3 * t] += B * (x[3 * k] - centre[0]);
            acc[3 * t + 1] += B * (x[3 * k + 1] - centre[1]);
            acc[3 * t + 2] += B * (x[3 * k + 2] - centre[2]);
        }
    }
}

/* oracle_step_coeffs with the external terms above included in F. */
void oracle_step_coeffs_ext(double *x, double *v, const double *m, int64_t n, double eps2, double G,
                            double d1, double cv, double ck, double d2,
                            double S, const double *x_psi, double rho_bar, const double *centre, double *work)
{
    int64_t i;
    for (i = 0; i < 3 * n; ++i) x[i] = x[i] + d1 * v[i];
    oracle_forces(x, m, n, eps2, G, NULL, n, work, NULL);
    oracle_add_external(x, NULL, n, eps2, S, x_psi, G, rho_bar, centre, work);
    for (i = 0; i < 3 * n; ++i) v[i] = cv * v[i] + ck * work[i];
    for (i = 0; i < 3 * n; ++i) x[i] = x[i] + d2 * v[i];
}

/* Eq. (2):  H(a) = H0 sqrt(Om_R a^-4 + Om_M a^-3 + Om_K a^-2 + Om_L). */
double oracle_hubble(double H0, double Om_R, double Om_M, double Om_K, double Om_L, double a)
{
    return H0 * sqrt(Om_R / (a * a * a * a) + Om_M / (a * a * a) + Om_K / (a * a) + Om_L);
}

/*
 * Integrate eq. (2) written as da/dt = a H(a) from a0 over a time interval dt
 * with classical RK4 and `substeps` equal sub-steps.
 */
double oracle_a_advance(double H0, double Om_R, double Om_M, double Om_K, double Om_L,
                        double a0, double dt, int substeps)
{
    const double h = dt / substeps;
    double a = a0;
    for (int s = 0; s < substeps; ++s) {
        const double k1 = a * oracle_hubble(H0, Om_R, Om_M, Om_K, Om_L, a);
        const double a2 = a + 0.5 * h * k1;
        const double k2 = a2 * oracle_hubble(H0, Om_R, Om_M, Om_K, Om_L, a2);
        const double a3 = a + 0.5 * h * k2;
        const double k3 = a3 * oracle_hubble(H0, Om_R, Om_M, Om_K, Om_L, a3);
        const double a4 = a + h * k3;
        const double k4 = a4 * oracle_hubble(H0, Om_R, Om_M, Om_K, Om_L, a4);
        a += h * (k1 + 2.0 * k2 + 2.0 * k3 + k4) / 6.0;
    }
    return a;
}

/*
 * Cosmic time since a = 0:  t(a) = integral_0^a da' / (a' H(a'))  (eq. 2 with
 * dt = da / (a H)).  Midpoint rule in the variable s = sqrt(a'), which removes
 * the integrable end-point behaviour of the matter and radiation eras:
 * da' = 2 s ds, so t = integral_0^sqrt(a) 2 ds / (s H(s^2)).
 */
double oracle_time_of_a(double H0, double Om_R, double Om_M, double Om_K, double Om_L,
                        double a, int64_t panels)
{
    const double smax = sqrt(a);
    const double h = smax / (double)panels;
    double sum = 0.0;
    for (int64_t i = 0; i < panels; ++i) {
        const double s = (i + 0.5) * h;
        sum += 2.0 / (s * oracle_hubble(H0, Om_R, Om_M, Om_K, Om_L, s * s));
    }
    return sum * h;
}

/*
 * integral_{t0}^{t0+dt} dt / a^p  along the solution of eq. (2) starting from
 * a(t0) = a0: the drift (p = 2) and kick (p = 1) integrals of eq. (9),
 * PAPER.md:64.  Composite Simpson in t with a(t) from oracle_a_advance.
 */
double oracle_int_dt_over_a_pow(double H0, double Om_R, double Om_M, double Om_K, double Om_L,
                                double a0, double dt, double p, int panels /* even */)
{
    const double h = dt / panels;
    double a = a0, sum = pow(a0, -p);
    for (int i = 1; i <= panels; ++i) {
        a = oracle_a_advance(H0, Om_R, Om_M, Om_K, Om_L, a, h, 8);
        const double f = pow(a, -p);
        sum += (i == panels) ? f : ((i & 1) ? 4.0 * f : 2.0 * f);
    }
    return sum * h / 3.0;
}

/*
 * Diagnostics of step a7 (canonical momentum p = m a^2 v and the
 * Hamiltonian of eq. (7)):
 *   out[0]      M  = sum m
 *   out[1..3]   P  = sum m v
 *   out[4..6]   a^2 P (canonical momentum sum)
 *   out[7]      T  = 1/2 sum m a^2 v^2
 *   out[8]      W  = -(G / 2a) sum_k sum_{j != k} m_k m_j / sqrt(r^2 + eps^2)   (NaN if !with_potential)
 *   out[9..11]  C  = sum m x / M
 */
void oracle_diagnostics(const double *x, const double *v, const double *m, int64_t n,
                        double eps2, double G, double a, int with_potential, double *out)
{
    double M = 0, P[3] = {0, 0, 0}, T = 0, C[3] = {0, 0, 0};
    for (int64_t k = 0; k < n; ++k) {
        M += m[k];
        for (int c = 0; c < 3; ++c) {
            P[c] += m[k] * v[3 * k + c];
            C[c] += m[k] * x[3 * k + c];
            T += 0.5 * m[k] * a * a * v[3 * k + c] * v[3 * k + c];
        }
    }
    out[0] = M;
    for (int c = 0; c < 3; ++c) { out[1 + c] = P[c]; out[4 + c] = a * a * P[c]; out[9 + c] = C[c] / M; }
    out[7] = T;
    if (with_potential) {
        double *acc = (double *)malloc(sizeof(double) * 3 * (size_t)n);
        double *phi = (double *)malloc(sizeof(double) * (size_t)n);
        oracle_forces(x, m, n, eps2, G, NULL, n, acc, phi);
        double W = 0;
        for (int64_t k = 0; k < n; ++k) W += 0.5 * m[k] * phi[k];
        out[8] = W / a;
        free(acc);
        free(phi);
    } else {
        out[8] = NAN;
    }
}

/*
 * Headless snapshot (NEXT row f4 of SURVEY 8f): the content of the paper's live
 * display, "other library shows a particle motion in the box" (PAPER.md:115,
 * App. A step 7) and of the Fig. 1 panels, as a particle-count
 * image.  The paper gives no rendering algorithm; reading G23:
 * orthographic projection along `axis`, one count per particle per pixel.
 *
 *   image axes (u, v) = the two other coordinates in cyclic order
 *       axis 0: u = y, v = z;   axis 1: u = z, v = x;   axis 2: u = x, v = y
 *   depth w = coordinate `axis`
 *   window = (u0, u1, v0, v1, w0, w1): a particle is counted iff  w0 <= w < w1
 *       and its pixel lies inside the image
 *   pixel, decided in FP32 -- the precision of the device state -- with every
 *   operation rounded once (this file is built with -ffp-contract=off):
 *       su = (float)width / (u1 - u0),   tu = (u - u0) * su,   pu = floor(tu)
 *       inside iff 0 <= tu < (float)width;       same for v with `height`
 *   image[pv * width + pu] += 1        (row-major, uint32, zeroed first)
 *
 * pos_mass: float [n][4] (x, y, z, m) -- the same FP32 array the GPU gets.
 * Pins (P14): brute force with exact rational arithmetic on dyadic inputs,
 * total = number of in-window particles, marginals = numpy.histogram.
 */
void oracle_splat(const float *pos_mass, int64_t n, int axis, const float *window,
                  int width, int height, uint32_t *image)
{
    const int iu = (axis + 1) % 3, iv = (axis + 2) % 3;
    const float u0 = window[0], u1 = window[1], v0 = window[2], v1 = window[3];
    const float w0 = window[4], w1 = window[5];
    const float su = (float)width / (u1 - u0);
    const float sv = (float)height / (v1 - v0);
    for (int64_t p = 0; p < (int64_t)width * height; ++p) image[p] = 0u;
    for (int64_t k = 0; k < n; ++k) {
        const float u = pos_mass[4 * k + iu], v = pos_mass[4 * k + iv], w = pos_mass[4 * k + axis];
        if (!(w >= w0 && w < w1)) continue;
        const float du = u - u0;
        const float tu = du * su;
        const float dv = v - v0;
        const float tv = dv * sv;
        if (!(tu >= 0.0f && tu < (float)width)) continue;
        if (!(tv >= 0.0f && tv < (float)height)) continue;
        const int pu = (int)floorf(tu), pv = (int)floorf(tv);
        image[(int64_t)pv * width + pu] += 1u;
    }
}

/*
 * Power spectrum of the velocity time series of each tracer particle (NEXT row
 * f3 of SURVEY 8f): the paper's stated purpose for following single particles,
 * "computation of the velocity of a single particle at every time-step ... and
 * its energy power spectrum".  The paper gives no formula; reading
 * G24: the periodogram of the recorded series, summed over the
 * three velocity components,
 *
 *   P_t[f] = (1/S) sum_{c=x,y,z} | sum_{s=0}^{S-1} v_{t,c}[s] exp(-2 pi i f s / S) |^2,
 *   f = 0 .. floor(S/2)                      (one-sided; real input)
 *
 * so that (Parseval)  sum over the full circle f = 0..S-1 of P_t[f] equals
 * sum_s |v_t[s]|^2  = twice the tracer's kinetic energy per unit mass summed
 * over the record.
 *
 * series: float [S][k][4] -- rows of the tracer ring, (vx, vy, vz, tag); the tag
 * is ignored.  out: double [k][S/2 + 1].  Direct O(k S^2) evaluation of the
 * definition; the phase is reduced exactly, (f s) mod S, before it is scaled.
 * Pins (P15): a pure sinusoid (S A^2 / 4 in its own bin), a constant (S c^2 in
 * bin 0), Parseval, and numpy.fft.rfft.
 */
void oracle_trace_spectrum(const float *series, int64_t S, int64_t k, double *out)
{
    const double two_pi = 6.283185307179586476925286766559;
    const int64_t nf = S / 2 + 1;
    int64_t t;
#pragma omp parallel for schedule(static)
    for (t = 0; t < k; ++t) {
        for (int64_t f = 0; f < nf; ++f) {
            double re[3] = {0, 0, 0}, im[3] = {0, 0, 0};
            for (int64_t s = 0; s < S; ++s) {
                const double ang = two_pi * (double)((f * s) % S) / (double)S;
                const double c = cos(ang), sn = sin(ang);
                for (int d = 0; d < 3; ++d) {
                    const double val = (double)series[(s * k + t) * 4 + d];
                    re[d] += val * c;
                    im[d] -= val * sn;
                }
            }
            out[t * nf + f] = (re[0] * re[0] + im[0] * im[0] + re[1] * re[1] + im[1] * im[1]
                               + re[2] * re[2] + im[2] * im[2]) / (double)S;
        }
    }
}
