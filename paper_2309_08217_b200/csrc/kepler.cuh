// kepler.cuh -- the per-body Kepler drift as a device function (see drift.cu for the derivation):
// universal variables, Stumpff series with argument quartering, Laguerre-Conway iteration.
#pragma once

#include "genga_internal.cuh"

namespace genga {

// c0..c3 at z: series for |z| <= 0.1 after quartering z, then the duplication formulae
//   c0(4z) = 2 c0^2 - 1, c1(4z) = c0 c1, c2(4z) = c1^2 / 2, c3(4z) = (c2 + c0 c3) / 4.
__device__ __forceinline__ void stumpff(double z, double& c0, double& c1, double& c2, double& c3)
{
    int k = 0;
    while (fabs(z) > 0.1 && k < 40) { z *= 0.25; ++k; }
    // c2 = sum (-z)^n / (2n+2)!,  c3 = sum (-z)^n / (2n+3)!   (n = 0..7)
    c2 = 1.0 / 20922789888000.0;                       // 1/16!
    c2 = fma(-z, c2, 1.0 / 87178291200.0);             // 1/14!
    c2 = fma(-z, c2, 1.0 / 479001600.0);               // 1/12!
    c2 = fma(-z, c2, 1.0 / 3628800.0);                 // 1/10!
    c2 = fma(-z, c2, 1.0 / 40320.0);                   // 1/8!
    c2 = fma(-z, c2, 1.0 / 720.0);                     // 1/6!
    c2 = fma(-z, c2, 1.0 / 24.0);                      // 1/4!
    c2 = fma(-z, c2, 0.5);                             // 1/2!
    c3 = 1.0 / 355687428096000.0;                      // 1/17!
    c3 = fma(-z, c3, 1.0 / 1307674368000.0);           // 1/15!
    c3 = fma(-z, c3, 1.0 / 6227020800.0);              // 1/13!
    c3 = fma(-z, c3, 1.0 / 39916800.0);                // 1/11!
    c3 = fma(-z, c3, 1.0 / 362880.0);                  // 1/9!
    c3 = fma(-z, c3, 1.0 / 5040.0);                    // 1/7!
    c3 = fma(-z, c3, 1.0 / 120.0);                     // 1/5!
    c3 = fma(-z, c3, 1.0 / 6.0);                       // 1/3!
    c1 = fma(-z, c3, 1.0);
    c0 = fma(-z, c2, 1.0);
    for (; k > 0; --k) {
        c3 = 0.25 * (c2 + c0 * c3);
        c2 = 0.5 * c1 * c1;
        c1 = c0 * c1;
        c0 = fma(2.0 * c0, c0, -1.0);
    }
}

// Propagate one body by dt_full about mu (in place).  Returns false if the iteration did not converge.
__device__ __forceinline__ bool kepler_drift(double mu, double dt_full, double& x0, double& y0, double& z0,
                                             double& vx, double& vy, double& vz)
{
    const double r0 = sqrt(x0 * x0 + y0 * y0 + z0 * z0);
    const double v2 = vx * vx + vy * vy + vz * vz;
    const double u  = x0 * vx + y0 * vy + z0 * vz;
    const double alpha = 2.0 * mu / r0 - v2;

    double dt = dt_full;
    if (alpha > 0.0) {                                   // closed orbit: drop whole revolutions
        const double P = 6.283185307179586476925286766559 * mu / (alpha * sqrt(alpha));
        if (fabs(dt) > 0.5 * P) dt = fma(-P, rint(dt / P), dt);
    }

    double s = dt / r0;                                  // first-order start
    {   // second-order refinement of the start (series of s in dt)
        const double a1 = u / (r0 * r0);
        s = s * (1.0 - 0.5 * a1 * s);
    }
    double c0 = 1, c1 = 1, c2 = 0.5, c3 = 1.0 / 6.0, G1 = 0, G2 = 0, r = r0;
    bool ok = false, last = false;
    for (int it = 0; it < 32; ++it) {
        stumpff(alpha * s * s, c0, c1, c2, c3);
        G1 = s * c1;
        G2 = s * s * c2;
        const double G3 = s * s * s * c3;
        const double t1 = r0 * G1, t2 = u * G2, t3 = mu * G3;
        const double F  = ((t1 + t2) + t3) - dt;
        r               = fma(r0, c0, fma(u, G1, mu * G2));
        if (last) { ok = true; break; }                  // previous step was the final one
        const double Fnoise = 4.0e-16 * (fabs(t1) + fabs(t2) + fabs(t3) + fabs(dt));
        const double Fpp  = fma(mu - alpha * r0, G1, u * c0);
        const double disc = fabs(16.0 * r * r - 20.0 * F * Fpp);
        const double den  = r + copysign(sqrt(disc), r);
        const double ds   = -5.0 * F / den;
        // converged: the step is below the resolution of s, or the residual is rounding noise
        if (!(fabs(ds) > 2.0e-15 * fabs(s)) || fabs(F) <= Fnoise) { ok = true; break; }
        s += ds;
        // the iteration converges at third order: after a step below 1e-8 |s| the next
        // correction is far below rounding, so only the G's are refreshed once more
        last = fabs(ds) < 1.0e-8 * fabs(s);
    }

    const double f  = 1.0 - mu * G2 / r0;
    const double g  = fma(r0, G1, u * G2);
    const double fd = -mu * G1 / (r * r0);
    const double gd = 1.0 - mu * G2 / r;
    const double nx = fma(f, x0, g * vx), ny = fma(f, y0, g * vy), nz = fma(f, z0, g * vz);
    const double wx = fma(fd, x0, gd * vx), wy = fma(fd, y0, gd * vy), wz = fma(fd, z0, gd * vz);
    x0 = nx; y0 = ny; z0 = nz; vx = wx; vy = wy; vz = wz;
    return ok;
}

}  // namespace genga
