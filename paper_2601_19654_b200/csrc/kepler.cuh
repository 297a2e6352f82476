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

// returns 0 ok / 1 failed (state untouched); *iters = Newton iterations used
__device__ __forceinline__ int drift_body(double mu, double dt_full, double& x, double& y, double& z, double& vx,
                                          double& vy, double& vz, int* iters) {
    const double r0 = sqrt(fma(z, z, fma(y, y, x * x)));
    *iters = 0;
    if (!(r0 > 0.0)) return 1;
    const double v2 = fma(vz, vz, fma(vy, vy, vx * vx));
    const double eta0 = fma(z, vz, fma(y, vy, x * vx));
    const double beta = 2.0 * mu / r0 - v2;
    // A bound orbit returns to the same state after T = 2 pi mu / beta^(3/2): drop whole
    // periods first.  Otherwise z = beta X^2 grows like (2 pi dt/T)^2, each argument
    // quartering of stumpff() doubles the phase error and dt - mu G3 cancels ~dt/T digits.
    double dt = dt_full;
    if (beta > 0.0) {
        const double T = 6.283185307179586 * mu / (beta * sqrt(beta));
        if (fabs(dt_full) > T) dt = fma(-rint(dt_full / T), T, dt_full);
    }
    double X = dt / r0;
    bool conv = false;
    int it = 0;
    for (; it < DRIFT_MAX_NEWTON; ++it) {
        const GF g = gfuncs(X, beta);
        const double F = fma(r0, g.G1, fma(eta0, g.G2, mu * g.G3)) - dt;
        const double r = fma(r0, g.G0, fma(eta0, g.G1, mu * g.G2));
        if (!(r > 0.0) || !isfinite(F)) break;
        const double dX = -F / r;
        X += dX;
        // quadratic convergence: a step below 1e-9 |X| leaves an error far below 1 ulp
        if (fabs(dX) <= 1e-9 * fabs(X) || dX == 0.0) { conv = true; ++it; break; }
    }
    *iters = it;
    if (!conv) {  // bisection on a bracket grown from 0 (F(0) = -dt, F monotone)
        const double sgn = dt >= 0.0 ? 1.0 : -1.0;
        double a = 0.0, b = sgn * fabs(dt / r0);
        bool ok = false;
        for (int k = 0; k < 128; ++k) {
            const GF g = gfuncs(b, beta);
            const double F = fma(r0, g.G1, fma(eta0, g.G2, mu * g.G3)) - dt;
            if (!isfinite(F)) return 1;
            if (F * sgn >= 0.0) { ok = true; break; }
            a = b; b *= 2.0;
        }
        if (!ok) return 1;
        for (int k = 0; k < 128; ++k) {
            const double m = 0.5 * (a + b);
            const GF g = gfuncs(m, beta);
            const double F = fma(r0, g.G1, fma(eta0, g.G2, mu * g.G3)) - dt;
            if (F * sgn >= 0.0) b = m; else a = m;
            if (fabs(b - a) <= 4.4e-16 * fabs(b)) break;
        }
        X = 0.5 * (a + b);
    }
    const GF g = gfuncs(X, beta);
    const double r = fma(r0, g.G0, fma(eta0, g.G1, mu * g.G2));
    if (!(r > 0.0)) return 1;
    const double fm1 = -mu * g.G2 / r0;
    const double gg = dt - mu * g.G3;
    const double fd = -mu * g.G1 / (r0 * r);
    const double gdm1 = -mu * g.G2 / r;
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
