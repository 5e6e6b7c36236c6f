// encounter.cuh -- NEXT-1 (reading R11), opt-in (params.encounter_mode = 1): the
// encounter complement of the hybrid symplectic step.  PAPER.md:45: "a changeover function smoothly switches"
// a pair between the fixed-step level-0 integrator and the close-encounter integrator; PAPER.md:55, 159:
// close-encounter pairs and groups; encounter forces always in double precision.
//
// During A(dt) a body that belongs to no encounter pair moves on its Kepler orbit (kepler.cuh).  The bodies of
// an encounter GROUP (a connected component of the pair list of the opening force evaluation) move under
//     H_A,group = sum_k (|p_k|^2 / 2 m_k - G M m_k / r_k) - sum_{k<l in group} G m_k m_l (1 - K(r_kl)) / r_kl,
// integrated in FP64 with classical RK4 substeps by ONE WARP per group, lane k holding member k's state in
// registers and reading the other members' stage positions by warp shuffles.  Pair weight (1 - K) + r K' (the complement of the kick's K - r K'); r_crit,kl held at the values
// of the opening force evaluation (w.rcrit / w.semi / w.vkep / w.m, API order).
#pragma once

#include "genga_internal.cuh"

namespace genga {
namespace enc {

constexpr int GMAX = 8;            // largest encounter group (members sit in lanes 0 .. n-1 of the group's warp)
constexpr int GINFO = GMAX + 1;    // ints per group in Workspace::ginfo: member count, members

using EncParams = EncArgs;

__device__ __forceinline__ double pair_rcrit(const EncParams& P, double mi, double mj, double rci, double rcj,
                                             double ai, double aj, double vki, double vkj)
{
    if (P.pair_rule == GENGA_PAIR_MUTUAL_HILL) {
        const double hill = P.n1 * cbrt((mi + mj) / (3.0 * P.M_star)) * (0.5 * (ai + aj));
        return fmax(hill, P.n2dt * fmax(vki, vkj));
    }
    return fmax(rci, rcj);
}

constexpr unsigned int FULL = 0xffffffffu;

__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(FULL, v, src); }

// 1/sqrt and 1/x from the MUFU seeds (rsqrt/rcp.approx.f64: about 2^-20 relative) with a cubic correction:
// relative error O(e^3) ~ 1e-18, i.e. a few ulp, at a fraction of the dependent latency of sqrt and divide.
__device__ __forceinline__ double rsq_seed(double a) { double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r; }
__device__ __forceinline__ double rcp_seed(double a) { double r; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r; }

// dv/dt of this lane's member at the stage positions (px, py, pz); every lane of the warp must call it.
// c01[l] = 0.1 r_crit,kl and i09[l] = 1 / (0.9 r_crit,kl) (0: no zone, the lane itself, an idle lane) for the
// members l.  NN > 0: the group size at compile time (straight-line code: the pair terms and the Kepler term
// overlap in the pipeline); NN = 0: n at run time.  Branch-free: a term that does not apply gets weight 0.
// CRIT: also return in tau the shortest time scale q / (|v_rel| + v_escape(q)) over the pairs of this member
// that are inside their zone (1e300 if none), from which the adaptive substep is taken (vx, vy, vz: own velocity).
template <int NN, bool CRIT = false>
__device__ __forceinline__ void member_accel(const EncParams& P, int n, double gm_self,
                                             const double (&c01)[GMAX], const double (&i09)[GMAX],
                                             double px, double py, double pz, double& a0, double& a1, double& a2,
                                             double vx = 0.0, double vy = 0.0, double vz = 0.0, double* tau = nullptr)
{
    double tmin = 1.0e300;
    {
        const double mu = P.G * P.M_star;
        const double r2 = fma(pz, pz, fma(py, py, px * px));
        const double y0 = rsq_seed(r2), t = y0 * y0, e = fma(-r2, t, 1.0), g = y0 * t;
        const double ir3 = -mu * fma(g * e, fma(1.875, e, 1.5), g);         // -mu / r^3
        a0 = px * ir3; a1 = py * ir3; a2 = pz * ir3;
    }
#pragma unroll
    for (int l = 0; l < (NN > 0 ? NN : GMAX); ++l) {
        if (NN == 0 && l >= n) break;                       // n is uniform over the warp
        const double ox = shfl_d(px, l), oy = shfl_d(py, l), oz = shfl_d(pz, l), ogm = shfl_d(gm_self, l);
        const double d0 = ox - px, d1 = oy - py, d2 = oz - pz;
        const double q2 = fma(d2, d2, fma(d1, d1, d0 * d0));
        const bool   on = (i09[l] > 0.0) && (q2 > 0.0);
        const double qs = on ? q2 : 1.0;
        const double y0 = rsq_seed(qs), t = y0 * y0, e = fma(-qs, t, 1.0), g = y0 * t;
        const double q0 = qs * y0;
        const double q  = fma(q0 * e, fma(0.375, e, 0.5), q0);              // |d|
        const double y  = fmin(fmax((q - c01[l]) * i09[l], 0.0), 1.0);       // y <= 0: Wc = 1, y >= 1: Wc = 0
        const double D  = fma(2.0 * y, y - 1.0, 1.0);                        // 2y^2 - 2y + 1, in [1/2, 1]
        const double r0 = rcp_seed(D), f = fma(-D, r0, 1.0);
        const double iD = fma(r0 * f, 1.0 + f, r0);
        const double K  = y * y * iD;
        const double Kp = 2.0 * y * (1.0 - y) * iD * iD * i09[l];            // dK/dr (0 at both ends)
        const double Wc = on ? 1.0 - (K - q * Kp) : 0.0;
        const double s  = ogm * Wc * fma(g * e, fma(1.875, e, 1.5), g);      // G m_l Wc / |d|^3
        a0 = fma(s, d0, a0); a1 = fma(s, d1, a1); a2 = fma(s, d2, a2);
        if (CRIT) {
            const double u0 = shfl_d(vx, l) - vx, u1 = shfl_d(vy, l) - vy, u2 = shfl_d(vz, l) - vz;
            const double vrel = sqrt(fma(u2, u2, fma(u1, u1, u0 * u0)));
            const double vesc = sqrt(2.0 * (gm_self + ogm) * y0);           // y0 ~ 1/|d| (seed accuracy is plenty here)
            if (on && y < 1.0) tmin = fmin(tmin, q / (vrel + vesc));
        }
    }
    if (CRIT) *tau = tmin;
}

// The flow of H_A,group over dt for this lane's member (state in registers): classical RK4 substeps of dt / nsub, or
// shorter where a pair is deep inside its zone (P.eta > 0: h = min(dt / nsub, eta * tau), tau the shortest
// q / (|v_rel| + v_escape) over the in-zone pairs of the whole group, never below dt / (256 nsub): status bit 8).
template <int NN, bool ADAPT>
__device__ __forceinline__ void integrate(const EncParams& P, int n, double gm, const double (&c01)[GMAX], const double (&i09)[GMAX],
                                          double dt, double& x0, double& x1, double& x2, double& v0, double& v1, double& v2,
                                          unsigned int* status)
{
    const double T = fabs(dt), sgn = (dt < 0.0) ? -1.0 : 1.0;
    const double hmax = T / P.nsub, hmin = hmax * (1.0 / 256.0);
    constexpr bool adaptive = ADAPT;
    double tnow = 0.0;
    bool floored = false;
    for (int s = 0; ; ++s) {
        if (adaptive ? !(T - tnow > 1.0e-9 * hmax) : (s == P.nsub)) break;
        double k0, k1, k2;                                 // stage acceleration
        double sx0, sx1, sx2, sv0, sv1, sv2;               // running sums k1 + 2 k2 + 2 k3 (+ k4)
        double t0, t1, t2, u0, u1, u2;                     // stage position, stage velocity
        double habs = hmax;
        if (adaptive) {
            double tau;
            member_accel<NN, true>(P, n, gm, c01, i09, x0, x1, x2, k0, k1, k2, v0, v1, v2, &tau);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) tau = fmin(tau, __shfl_xor_sync(FULL, tau, o));
            const double want = P.eta * tau;
            if (want < hmin) floored = true;
            habs = fmin(hmax, fmax(want, hmin));
            habs = fmin(habs, T - tnow);
            tnow += habs;
        } else {
            member_accel<NN>(P, n, gm, c01, i09, x0, x1, x2, k0, k1, k2);
        }
        const double h = sgn * habs, hh = 0.5 * h, h6 = h / 6.0;
        sx0 = v0; sx1 = v1; sx2 = v2; sv0 = k0; sv1 = k1; sv2 = k2;
        t0 = fma(hh, v0, x0); t1 = fma(hh, v1, x1); t2 = fma(hh, v2, x2);
        u0 = fma(hh, k0, v0); u1 = fma(hh, k1, v1); u2 = fma(hh, k2, v2);
        member_accel<NN>(P, n, gm, c01, i09, t0, t1, t2, k0, k1, k2);
        sx0 += 2.0 * u0; sx1 += 2.0 * u1; sx2 += 2.0 * u2; sv0 += 2.0 * k0; sv1 += 2.0 * k1; sv2 += 2.0 * k2;
        t0 = fma(hh, u0, x0); t1 = fma(hh, u1, x1); t2 = fma(hh, u2, x2);
        u0 = fma(hh, k0, v0); u1 = fma(hh, k1, v1); u2 = fma(hh, k2, v2);
        member_accel<NN>(P, n, gm, c01, i09, t0, t1, t2, k0, k1, k2);
        sx0 += 2.0 * u0; sx1 += 2.0 * u1; sx2 += 2.0 * u2; sv0 += 2.0 * k0; sv1 += 2.0 * k1; sv2 += 2.0 * k2;
        t0 = fma(h, u0, x0); t1 = fma(h, u1, x1); t2 = fma(h, u2, x2);
        u0 = fma(h, k0, v0); u1 = fma(h, k1, v1); u2 = fma(h, k2, v2);
        member_accel<NN>(P, n, gm, c01, i09, t0, t1, t2, k0, k1, k2);
        x0 = fma(h6, sx0 + u0, x0); x1 = fma(h6, sx1 + u1, x1); x2 = fma(h6, sx2 + u2, x2);
        v0 = fma(h6, sv0 + k0, v0); v1 = fma(h6, sv1 + k1, v1); v2 = fma(h6, sv2 + k2, v2);
    }
    if (floored && (threadIdx.x & 31) == 0) atomicOr(status, 8u);
}

// One warp advances group g through S(dt/2) (the shift s, already scaled) and the flow of H_A,group over dt
// (nsub RK4 substeps) and writes its members back.  Members are taken in ascending body index, so the result
// does not depend on the order in which group_kernel registered them.
__device__ __forceinline__ void warp_group(const EncParams& P, Workspace& w, int g, double dt, double s0, double s1, double s2)
{
    const int lane = threadIdx.x & 31;
    const int* info = w.ginfo + (size_t)g * GINFO;
    const int n = min(info[0], GMAX);
    const int b_in = (lane < n) ? info[1 + lane] : 0x7fffffff;
    int rank = 0;
#pragma unroll
    for (int l = 0; l < GMAX; ++l) { const int o = __shfl_sync(FULL, b_in, l); if (l < n && o < b_in) ++rank; }
    int b = -1;
#pragma unroll
    for (int l = 0; l < GMAX; ++l) {
        const int o = __shfl_sync(FULL, b_in, l), r = __shfl_sync(FULL, rank, l);
        if (l < n && r == lane) b = o;
    }
    const bool active = lane < n;
    double m = 0.0, rci = 0.0, sa = 0.0, vk = 0.0;
    double x0 = 1.0, x1 = 0.0, x2 = 0.0, v0 = 0.0, v1 = 0.0, v2 = 0.0;      // idle lanes: a harmless unit orbit
    if (active) {
        m = w.m[b]; rci = w.rcrit[b]; sa = w.semi[b]; vk = w.vkep[b];
        x0 = w.x[3 * b] + s0; x1 = w.x[3 * b + 1] + s1; x2 = w.x[3 * b + 2] + s2;
        v0 = w.v[3 * b]; v1 = w.v[3 * b + 1]; v2 = w.v[3 * b + 2];
    }
    double c01[GMAX], i09[GMAX];
#pragma unroll
    for (int l = 0; l < GMAX; ++l) {
        const double ml = shfl_d(m, l), rcl = shfl_d(rci, l), sal = shfl_d(sa, l), vkl = shfl_d(vk, l);
        const double rc = (active && l < n && l != lane) ? pair_rcrit(P, m, ml, rci, rcl, sa, sal, vk, vkl) : 0.0;
        c01[l] = 0.1 * rc; i09[l] = (rc > 0.0) ? 1.0 / (0.9 * rc) : 0.0;
    }
    const double gm = P.G * m;
    if (dt != 0.0) {
        unsigned int* st = &w.ctr->enc_status;
        if (P.eta > 0.0) {                                  // adaptive substeps (opt-in): one generic instance
            integrate<0, true>(P, n, gm, c01, i09, dt, x0, x1, x2, v0, v1, v2, st);
        } else {
            if (n == 2)      integrate<2, false>(P, n, gm, c01, i09, dt, x0, x1, x2, v0, v1, v2, st);
            else if (n == 3) integrate<3, false>(P, n, gm, c01, i09, dt, x0, x1, x2, v0, v1, v2, st);
            else if (n == 4) integrate<4, false>(P, n, gm, c01, i09, dt, x0, x1, x2, v0, v1, v2, st);
            else             integrate<0, false>(P, n, gm, c01, i09, dt, x0, x1, x2, v0, v1, v2, st);
        }
    }
    if (active) {
        w.x[3 * b] = x0; w.x[3 * b + 1] = x1; w.x[3 * b + 2] = x2;
        w.v[3 * b] = v0; w.v[3 * b + 1] = v1; w.v[3 * b + 2] = v2;
    }
}

}  // namespace enc
}  // namespace genga
