// drift.cu -- per-body heliocentric Kepler drift in FP64 with universal-variable f and g
// ("the Kepler orbit solver is always performed in double precision"; reading G4:
// the exact two-body map about mu = G M_star).
//
// With r0 = |x0|, u = x0.v0, alpha = 2 mu/r0 - |v0|^2 and the Stumpff functions c_k(z),
// G_k = s^k c_k(alpha s^2), the universal Kepler equation is
//     F(s) = r0 G1 + u G2 + mu G3 - dt = 0,   F' = r = r0 c0 + u G1 + mu G2,
//     F'' = (mu - alpha r0) G1 + u c0,
// solved by Laguerre-Conway iteration (n = 5).  Then
//     f = 1 - mu G2 / r0,  g = r0 G1 + u G2 (= dt - mu G3),  fdot = -mu G1 / (r r0),  gdot = 1 - mu G2 / r.
// This is a different formulation from the oracle's eccentric-anomaly-difference form on purpose.
#include "genga_internal.cuh"
#include "kepler.cuh"
#include "momentum.cuh"

namespace genga {

namespace {

constexpr int DRIFT_NT = 128;

__global__ void __launch_bounds__(DRIFT_NT)
drift_kernel(int N, double mu, double dt_full, double* __restrict__ x, double* __restrict__ v, Counters* ctr)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N || dt_full == 0.0) return;
    double x0 = x[3 * i], y0 = x[3 * i + 1], z0 = x[3 * i + 2];
    double vx = v[3 * i], vy = v[3 * i + 1], vz = v[3 * i + 2];
    if (!kepler_drift(mu, dt_full, x0, y0, z0, vx, vy, vz)) atomicAdd(&ctr->noconv, 1u);
    x[3 * i] = x0; x[3 * i + 1] = y0; x[3 * i + 2] = z0;
    v[3 * i] = vx; v[3 * i + 1] = vy; v[3 * i + 2] = vz;
}

// The middle of a fused step: Sun-kick S(tau_pre) with the momentum in mom[SLOT_A] (O8), Kepler drift
// D(dt) (O9), and the momentum of the drifted velocities into mom[SLOT_B] for the closing Sun-kick,
// which the next prep kernel applies.
__global__ void __launch_bounds__(DRIFT_NT)
shift_drift_mom_kernel(int N, double mu, double dt_full, double shift_scale, double* __restrict__ x,
                       double* __restrict__ v, const double* __restrict__ m, double* __restrict__ mom, Counters* ctr)
{
    const int i = blockIdx.x * DRIFT_NT + threadIdx.x;
    double p0 = 0, p1 = 0, p2 = 0, mt = 0;
    if (i < N) {
        double x0 = fma(shift_scale, mom[MOM_SLOT_A + 0], x[3 * i]);
        double y0 = fma(shift_scale, mom[MOM_SLOT_A + 1], x[3 * i + 1]);
        double z0 = fma(shift_scale, mom[MOM_SLOT_A + 2], x[3 * i + 2]);
        double vx = v[3 * i], vy = v[3 * i + 1], vz = v[3 * i + 2];
        if (dt_full != 0.0) {
            if (!kepler_drift(mu, dt_full, x0, y0, z0, vx, vy, vz)) atomicAdd(&ctr->noconv, 1u);
            v[3 * i] = vx; v[3 * i + 1] = vy; v[3 * i + 2] = vz;
        }
        x[3 * i] = x0; x[3 * i + 1] = y0; x[3 * i + 2] = z0;
        const double mi = m[i];
        p0 = mi * vx; p1 = mi * vy; p2 = mi * vz; mt = mi;
    }
    grid_momentum(p0, p1, p2, mt, mom + MOM_PARTIALS, mom + MOM_SLOT_B, &ctr->ticket);
}

}  // namespace

void launch_drift(const Handle* h, double dt)
{
    if (h->N == 0) return;
    drift_kernel<<<(h->N + 127) / 128, 128, 0, h->stream>>>(h->N, h->p.G * h->p.M_star, dt, h->w.x, h->w.v, h->w.ctr);
}

void launch_shift_drift_mom(const Handle* h, double tau_pre, double dt)
{
    if (h->N == 0) return;
    shift_drift_mom_kernel<<<(h->N + DRIFT_NT - 1) / DRIFT_NT, DRIFT_NT, 0, h->stream>>>(
        h->N, h->p.G * h->p.M_star, dt, tau_pre / h->p.M_star, h->w.x, h->w.v, h->w.m, h->w.mom, h->w.ctr);
}

}  // namespace genga
