// kepler.cuh - per-body Kepler drift about the star (arxes_drift, PAPER.md:59, 130,
// 231-233), Gauss f,g in universal variables:
//   c_n(z) = sum_k (-z)^k / (2k+n)! ,  G_n = X^n c_n(beta X^2),  beta = 2 mu / r0 - v0^2
//   solve  r0 G1 + eta0 G2 + mu G3 = dt   (d/dX = r = r0 G0 + eta0 G1 + mu G2 > 0)
//   x = x0 + (f-1) x0 + g v0,  v = v0 + fdot x0 + (gdot-1) v0
//   f-1 = -mu G2 / r0, g = dt - mu G3, fdot = -mu G1 / (r0 r), gdot-1 = -mu G2 / r
// One thread per body, FP64 throughout.
#pragma once
#include "common.cuh"

namespace mopal {

// c2, c3 for |z| <= 0.1 by an 8-term Taylor polynomial (truncation < 1e-22), larger |z|
// by quartering the argument and undoing it with the duplication formulas.
__device__ __forceinline__ void stumpff(double z, double& c0, double& c1, double& c2, double& c3) {
    int n = 0;
    while (fabs(z) > 0.1) { z *= 0.25; ++n; }
    // 1/(2k+2)! and 1/(2k+3)!, k = 0..7
    double a2 = 1.0 / 6402373705728000.0;   // 1/18!  (k = 8 guard term)
    double a3 = 1.0 / 121645100408832000.0; // 1/19!
    a2 = fma(-z, a2, 1.0 / 20922789888000.0);   // 1/16!
    a3 = fma(-z, a3, 1.0 / 355687428096000.0);  // 1/17!
    a2 = fma(-z, a2, 1.0 / 87178291200.0);      // 1/14!
    a3 = fma(-z, a3, 1.0 / 1307674368000.0);    // 1/15!
    a2 = fma(-z, a2, 1.0 / 479001600.0);        // 1/12!
    a3 = fma(-z, a3, 1.0 / 6227020800.0);       // 1/13!
    a2 = fma(-z, a2, 1.0 / 3628800.0);          // 1/10!
    a3 = fma(-z, a3, 1.0 / 39916800.0);         // 1/11!
    a2 = fma(-z, a2, 1.0 / 40320.0);            // 1/8!
    a3 = fma(-z, a3, 1.0 / 362880.0);           // 1/9!
    a2 = fma(-z, a2, 1.0 / 720.0);              // 1/6!
    a3 = fma(-z, a3, 1.0 / 5040.0);             // 1/7!
    a2 = fma(-z, a2, 1.0 / 24.0);               // 1/4!
    a3 = fma(-z, a3, 1.0 / 120.0);              // 1/5!
    a2 = fma(-z, a2, 0.5);                      // 1/2!
    a3 = fma(-z, a3, 1.0 / 6.0);                // 1/3!
    c2 = a2; c3 = a3;
    c1 = fma(-z, c3, 1.0);
    c0 = fma(-z, c2, 1.0);
    for (; n > 0; --n) {
        c3 = 0.25 * fma(c0, c3, c2);
        c2 = 0.5 * c1 * c1;
        c1 = c0 * c1;
        c0 = fma(2.0 * c0, c0, -1.0);
    }
}

struct GF { double G0, G1, G2, G3; };

__device__ __forceinline__ GF gfuncs(double X, double beta) {
    double c0, c1, c2, c3;
    const double X2 = X * X;
    stumpff(beta * X2, c0, c1, c2, c3);
    GF g;
    g.G0 = c0; g.G1 = X * c1; g.G2 = X2 * c2; g.G3 = X2 * X * c3;
    return g;
}

constexpr int DRIFT_MAX_NEWTON = 12;

// 1/sqrt(a) to ~1e-19 relative before rounding: MUFU.RSQ64H seed + one third-order correction
__device__ __forceinline__ double rsqrt_full(double a) {
    const double y = rsqrt_seed(a);
    const double e = fma(-a, y * y, 1.0);
    return fma(y * e, fma(0.375, e, 0.5), y);
}
// 1/a to ~1 ulp: MUFU.RCP64H seed + two Newton steps (no IEEE division sequence)
__device__ __forceinline__ double rcp_fast(double a) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double e = fma(-a, y, 1.0);
    y = fma(y, e, y);
    e = fma(-a, y, 1.0);
    return fma(y, e, y);
}

// returns 0 ok / 1 failed (state untouched); *iters = Newton iterations used
//
// Cost matters here: at ~500 FP64 instructions per body the kernel is FP64-issue bound, not HBM
// bound (96 B per body).  So: the start value is the third-order series inverse of Kepler's equation
// in X (exact for circular orbits, ~1e-6 relative for the disks' e ~ 0.02), a Newton step is
// accepted as final as soon as the leading-order error estimate of the NEXT iterate,
// |r'/(2r)| dX^2, is below 2e-16 |X| (normally the first step), and the G functions at the final X
// come from their Taylor expansion about the last evaluation point (dG3 = G2, dG2 = G1, dG1 = G0,
// dG0 = -beta G1; third order, error ~ dX^4) instead of another series evaluation.
__device__ __forceinline__ int drift_body(double mu, double dt_full, double& x, double& y, double& z, double& vx,
                                          double& vy, double& vz, int* iters) {
    const double r2 = fma(z, z, fma(y, y, x * x));
    *iters = 0;
    if (!(r2 > 0.0) || !isfinite(r2)) return 1;
    const double ir0 = rsqrt_full(r2);
    const double r0 = r2 * ir0;
    const double v2 = fma(vz, vz, fma(vy, vy, vx * vx));
    const double eta0 = fma(z, vz, fma(y, vy, x * vx));
    const double beta = fma(2.0 * mu, ir0, -v2);
    const double kappa = fma(-beta, r0, mu);          // mu - beta r0 = d^2 r / dX^2 at X = 0
    // A bound orbit returns to the same state after T = 2 pi mu / beta^(3/2): drop whole
    // periods first.  Otherwise z = beta X^2 grows like (2 pi dt/T)^2, each argument
    // quartering of stumpff() doubles the phase error and dt - mu G3 cancels ~dt/T digits.
    double dt = dt_full;
    if (beta > 0.0 && dt_full * dt_full * beta * beta * beta > 39.47841760435743 * mu * mu) {   // |dt| > T
        const double T = 6.283185307179586 * mu / (beta * sqrt(beta));
        dt = fma(-rint(dt_full / T), T, dt_full);
    }
    // dt = r0 X + eta0 X^2/2 + kappa X^3/6 + ...  inverted to third order in tau = dt / r0
    const double tau = dt * ir0;
    const double b1 = -0.5 * eta0 * ir0;
    const double c1 = fma(0.5 * eta0 * ir0, eta0, kappa * (-1.0 / 6.0)) * ir0;
    double X = tau * fma(tau, fma(tau, c1, b1), 1.0);
    if (!isfinite(X) || fabs(tau * fma(tau, c1, b1)) > 0.5) X = tau;   // series useless (large step): plain first order
    bool conv = false;
    int it = 0;
    GF g;
    double r = 0.0;
    for (; it < DRIFT_MAX_NEWTON; ++it) {
        g = gfuncs(X, beta);
        const double F = fma(r0, g.G1, fma(eta0, g.G2, mu * g.G3)) - dt;
        r = fma(r0, g.G0, fma(eta0, g.G1, mu * g.G2));
        if (!(r > 0.0) || !isfinite(F)) break;
        const double ir = rcp_fast(r);
        const double dX = -F * ir;
        const double Xn = X + dX;
        const double rp = fma(eta0, g.G0, kappa * g.G1);          // dr/dX
        // error of Xn to leading order: |r'/(2r)| dX^2; trust the estimate only for small steps
        if ((fabs(rp * ir) * dX * dX <= 4.0e-16 * fabs(Xn) && fabs(dX) <= 1e-3 * fabs(Xn)) || dX == 0.0) {
            // G_n(X + dX) by Taylor expansion about X
            const double h = 0.5 * dX, t3 = dX * (1.0 / 3.0);
            const double G3 = fma(dX, fma(h, fma(t3, g.G0, g.G1), g.G2), g.G3);
            const double G2 = fma(dX, fma(h, fma(-t3 * beta, g.G1, g.G0), g.G1), g.G2);
            const double G1 = fma(dX, fma(-h * beta, fma(t3, g.G0, g.G1), g.G0), g.G1);
            const double G0 = fma(-dX * beta, fma(h, fma(-t3 * beta, g.G1, g.G0), g.G1), g.G0);
            g.G0 = G0; g.G1 = G1; g.G2 = G2; g.G3 = G3;
            X = Xn;
            conv = true; ++it;
            break;
        }
        X = Xn;
    }
    *iters = it;
    if (!conv) {  // bisection on a bracket grown from 0 (F(0) = -dt, F monotone)
        const double sgn = dt >= 0.0 ? 1.0 : -1.0;
        double a = 0.0, b = sgn * fabs(dt * ir0);
        bool ok = false;
        for (int k = 0; k < 128; ++k) {
            const GF q = gfuncs(b, beta);
            const double F = fma(r0, q.G1, fma(eta0, q.G2, mu * q.G3)) - dt;
            if (!isfinite(F)) return 1;
            if (F * sgn >= 0.0) { ok = true; break; }
            a = b; b *= 2.0;
        }
        if (!ok) return 1;
        for (int k = 0; k < 128; ++k) {
            const double m = 0.5 * (a + b);
            const GF q = gfuncs(m, beta);
            const double F = fma(r0, q.G1, fma(eta0, q.G2, mu * q.G3)) - dt;
            if (F * sgn >= 0.0) b = m; else a = m;
            if (fabs(b - a) <= 4.4e-16 * fabs(b)) break;
        }
        X = 0.5 * (a + b);
        g = gfuncs(X, beta);
    }
    r = fma(r0, g.G0, fma(eta0, g.G1, mu * g.G2));
    if (!(r > 0.0)) return 1;
    const double ir = rcp_fast(r);
    const double mG2 = -mu * g.G2;
    const double fm1 = mG2 * ir0;
    const double gg = fma(-mu, g.G3, dt);
    const double fd = -mu * g.G1 * ir0 * ir;
    const double gdm1 = mG2 * ir;
    const double nx = x + fma(fm1, x, gg * vx);
    const double ny = y + fma(fm1, y, gg * vy);
    const double nz = z + fma(fm1, z, gg * vz);
    const double nvx = vx + fma(fd, x, gdm1 * vx);
    const double nvy = vy + fma(fd, y, gdm1 * vy);
    const double nvz = vz + fma(fd, z, gdm1 * vz);
    x = nx; y = ny; z = nz; vx = nvx; vy = nvy; vz = nvz;
    return 0;
}

}  // namespace mopal
