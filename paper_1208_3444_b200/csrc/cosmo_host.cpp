// cosmo_host.cpp -- host-only FP64 Friedmann helpers of libcolatus (eq. (2)).
//
//   da/dt = a H(a),   H(a) = H0 sqrt(Om_R a^-4 + Om_M a^-3 + Om_K a^-2 + Om_L)
//
// north_star: "Scale-factor integration is done on the host in double."  These routines use an
// adaptive Dormand-Prince 5(4) integrator and Gauss-Legendre quadrature; they share no code with
// the oracle's fixed-step RK4 / midpoint rule (oracle/colatus_oracle.c).
#include <cmath>
#include <limits>

#include "../../include/colatus.h"

namespace {

inline double hub(const colatus_cosmo *c, double a) {
    const double ia = 1.0 / a;
    return c->H0 * std::sqrt(((c->Om_R * ia + c->Om_M) * ia + c->Om_K) * ia * ia + c->Om_L);
}

// y = (a, I) with dI/dt = a^-p (p < 0 disables the second component)
struct Deriv {
    const colatus_cosmo *c;
    double p;
    inline void operator()(const double y[2], double f[2]) const {
        f[0] = y[0] * hub(c, y[0]);
        f[1] = (p >= 0.0) ? std::pow(y[0], -p) : 0.0;
    }
};

// Dormand-Prince 5(4) with step-size control on both components; integrates over `dt` (either sign).
// If the interval cannot be completed (step size underflows, e.g. a reaches 0 when integrating backwards, or
// the step guard is exhausted) both components are set to NaN: callers fail loudly instead of using a
// partial result.
void dopri(const Deriv &F, double y[2], double dt) {
    static const double c2 = 1.0 / 5, c3 = 3.0 / 10, c4 = 4.0 / 5, c5 = 8.0 / 9;
    static const double a21 = 1.0 / 5;
    static const double a31 = 3.0 / 40, a32 = 9.0 / 40;
    static const double a41 = 44.0 / 45, a42 = -56.0 / 15, a43 = 32.0 / 9;
    static const double a51 = 19372.0 / 6561, a52 = -25360.0 / 2187, a53 = 64448.0 / 6561, a54 = -212.0 / 729;
    static const double a61 = 9017.0 / 3168, a62 = -355.0 / 33, a63 = 46732.0 / 5247, a64 = 49.0 / 176,
                        a65 = -5103.0 / 18656;
    static const double b1 = 35.0 / 384, b3 = 500.0 / 1113, b4 = 125.0 / 192, b5 = -2187.0 / 6784, b6 = 11.0 / 84;
    static const double e1 = 71.0 / 57600, e3 = -71.0 / 16695, e4 = 71.0 / 1920, e5 = -17253.0 / 339200,
                        e6 = 22.0 / 525, e7 = -1.0 / 40;
    (void)c2; (void)c3; (void)c4; (void)c5;   // autonomous system: the nodes are not needed
    const double rtol = 1e-13;
    const double dir = (dt >= 0) ? 1.0 : -1.0;
    // first trial step: the whole interval, but no more than a tenth of the Hubble time at the start (the natural
    // scale of eq. (2)); the controller below shrinks or grows it from there.  A leapfrog half step is << 1/H, so the
    // per-step schedule of colatus_run costs one accepted step per call (it used to start at dt/16: 16 steps per
    // call, 1.5 us per leapfrog step -- a tenth of a whole N = 4096 step spent on the host before the first launch)
    double t = 0.0, h = dt;
    {
        double f0[2];
        F(y, f0);
        const double rate = std::fabs(f0[0]) / std::fmax(std::fabs(y[0]), 1e-300);      // |da/dt| / a = H
        if (std::isfinite(rate) && rate > 0.0 && std::fabs(h) * rate > 0.1) h = dir * 0.1 / rate;
    }
    double k1[2], k2[2], k3[2], k4[2], k5[2], k6[2], k7[2], w[2], ynew[2];
    int guard = 0;
    while ((dt - t) * dir > 0 && guard++ < 1000000) {
        if ((t + h - dt) * dir > 0) h = dt - t;
        F(y, k1);
        for (int i = 0; i < 2; ++i) w[i] = y[i] + h * a21 * k1[i];
        F(w, k2);
        for (int i = 0; i < 2; ++i) w[i] = y[i] + h * (a31 * k1[i] + a32 * k2[i]);
        F(w, k3);
        for (int i = 0; i < 2; ++i) w[i] = y[i] + h * (a41 * k1[i] + a42 * k2[i] + a43 * k3[i]);
        F(w, k4);
        for (int i = 0; i < 2; ++i) w[i] = y[i] + h * (a51 * k1[i] + a52 * k2[i] + a53 * k3[i] + a54 * k4[i]);
        F(w, k5);
        for (int i = 0; i < 2; ++i)
            w[i] = y[i] + h * (a61 * k1[i] + a62 * k2[i] + a63 * k3[i] + a64 * k4[i] + a65 * k5[i]);
        F(w, k6);
        for (int i = 0; i < 2; ++i)
            ynew[i] = y[i] + h * (b1 * k1[i] + b3 * k3[i] + b4 * k4[i] + b5 * k5[i] + b6 * k6[i]);
        F(ynew, k7);
        double err = 0.0;
        for (int i = 0; i < 2; ++i) {
            const double e = h * (e1 * k1[i] + e3 * k3[i] + e4 * k4[i] + e5 * k5[i] + e6 * k6[i] + e7 * k7[i]);
            const double sc = rtol * std::fmax(std::fabs(y[i]), std::fabs(ynew[i])) + 1e-300;
            err = std::fmax(err, std::fabs(e) / sc);
        }
        if (!(ynew[0] > 0.0) || !std::isfinite(ynew[0])) err = 1e30;   // stepped through a = 0: shrink
        if (err <= 1.0) {
            t += h;
            y[0] = ynew[0];
            y[1] = ynew[1];
        }
        const double fac = (err > 0.0) ? 0.9 * std::pow(err, -0.2) : 5.0;
        h *= std::fmin(5.0, std::fmax(0.1, fac));
        if (std::fabs(h) < 1e-300) break;
    }
    if ((dt - t) * dir > 0) y[0] = y[1] = std::numeric_limits<double>::quiet_NaN();
}

}  // namespace

extern "C" double colatus_hubble(const colatus_cosmo *c, double a) {
    if (!c || !(a > 0.0)) return std::numeric_limits<double>::quiet_NaN();
    return hub(c, a);
}

extern "C" double colatus_a_advance(const colatus_cosmo *c, double a0, double dt) {
    if (!c || !(a0 > 0.0) || !std::isfinite(dt)) return std::numeric_limits<double>::quiet_NaN();
    double y[2] = {a0, 0.0};
    dopri(Deriv{c, -1.0}, y, dt);
    return y[0];
}

extern "C" double colatus_int_dt_over_a_pow(const colatus_cosmo *c, double a0, double dt, double p) {
    if (!c || !(a0 > 0.0) || !std::isfinite(dt) || !(p >= 0.0)) return std::numeric_limits<double>::quiet_NaN();
    double y[2] = {a0, 0.0};
    dopri(Deriv{c, p}, y, dt);
    return y[1];
}

// t(a) = int_0^a da'/(a' H(a')).  With a' = u^2:  t = int_0^sqrt(a) 2 du / (u H(u^2)); the integrand
// is smooth at u = 0 for radiation (~u^3), matter (~u^2) and curvature (~u) dominated starts.
// Composite 8-point Gauss-Legendre on 256 panels.
extern "C" double colatus_time_of_a(const colatus_cosmo *c, double a) {
    if (!c || !(a > 0.0)) return std::numeric_limits<double>::quiet_NaN();
    if (c->Om_R == 0.0 && c->Om_M == 0.0 && c->Om_K == 0.0) return std::numeric_limits<double>::infinity();
    static const double xg[4] = {0.1834346424956498, 0.5255324099163290, 0.7966664774136267, 0.9602898564975363};
    static const double wg[4] = {0.3626837833783620, 0.3137066458778873, 0.2223810344533745, 0.1012285362903763};
    const int panels = 256;
    const double umax = std::sqrt(a), hp = umax / panels;
    double sum = 0.0;
    for (int i = 0; i < panels; ++i) {
        const double mid = (i + 0.5) * hp;
        for (int g = 0; g < 4; ++g)
            for (int sgn = -1; sgn <= 1; sgn += 2) {
                const double u = mid + sgn * 0.5 * hp * xg[g];
                sum += wg[g] * 2.0 / (u * hub(c, u * u));
            }
    }
    return sum * 0.5 * hp;
}
