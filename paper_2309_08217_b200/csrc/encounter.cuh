// encounter.cuh -- NEXT-1 (reading R11), opt-in (params.encounter_mode = 1): the
// encounter complement of the hybrid symplectic step.  PAPER.md:45: "a changeover function smoothly switches"
// a pair between the fixed-step level-0 integrator and the close-encounter integrator; PAPER.md:55, 159:
// close-encounter pairs and groups; encounter forces always in double precision.
//
// During A(dt) a body that belongs to no encounter pair moves on its Kepler orbit (kepler.cuh).  The bodies of
// an encounter GROUP (a connected component of the pair list of the opening force evaluation) move under
//     H_A,group = sum_k (|p_k|^2 / 2 m_k - G M m_k / r_k) - sum_{k<l in group} G m_k m_l (1 - K(r_kl)) / r_kl,
// integrated in FP64 with classical RK4 substeps by the thread of the group's leader (its smallest body
// index).  Pair weight (1 - K) + r K' (the complement of the kick's K - r K'); r_crit,kl held at the values
// of the opening force evaluation (w.rcrit / w.semi / w.vkep / w.m, API order).
#pragma once

#include "genga_internal.cuh"

namespace genga {
namespace enc {

constexpr int GMAX = 8;            // largest encounter group the leader thread integrates

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

// complement weight 1 - (K - r K') = (1 - K) + r K'
__device__ __forceinline__ double weight_c(double r, double rc)
{
    if (!(rc > 0.0)) return (r > 0.0) ? 0.0 : 1.0;
    const double y = (r - 0.1 * rc) / (0.9 * rc);
    if (y <= 0.0) return 1.0;
    if (y >= 1.0) return 0.0;
    const double D = 2.0 * y * y - 2.0 * y + 1.0;
    const double K = (y * y) / D;
    return 1.0 - (K - r * ((2.0 * y * (1.0 - y) / (D * D)) / (0.9 * rc)));
}

struct GroupState { int n; int body[GMAX]; double m[GMAX]; double x[GMAX][3]; double v[GMAX][3]; double rc[GMAX][GMAX]; };

__device__ __forceinline__ void group_rhs(const EncParams& P, const GroupState& g, const double (*x)[3], const double (*v)[3],
                                          double (*dx)[3], double (*dv)[3])
{
    const double mu = P.G * P.M_star;
    for (int k = 0; k < g.n; ++k) {
        const double r2 = x[k][0] * x[k][0] + x[k][1] * x[k][1] + x[k][2] * x[k][2];
        const double ir3 = 1.0 / (r2 * sqrt(r2));
        double a0 = -mu * x[k][0] * ir3, a1 = -mu * x[k][1] * ir3, a2 = -mu * x[k][2] * ir3;
        for (int l = 0; l < g.n; ++l) {
            if (l == k) continue;
            const double d0 = x[l][0] - x[k][0], d1 = x[l][1] - x[k][1], d2 = x[l][2] - x[k][2];
            const double q2 = d0 * d0 + d1 * d1 + d2 * d2;
            const double q = sqrt(q2);
            if (!(q > 0.0)) continue;
            const double Wc = weight_c(q, g.rc[k][l]);
            if (Wc == 0.0) continue;
            const double s = P.G * g.m[l] * Wc / (q2 * q);
            a0 = fma(s, d0, a0); a1 = fma(s, d1, a1); a2 = fma(s, d2, a2);
        }
        dx[k][0] = v[k][0]; dx[k][1] = v[k][1]; dx[k][2] = v[k][2];
        dv[k][0] = a0; dv[k][1] = a1; dv[k][2] = a2;
    }
}

// nsub RK4 substeps of the flow of H_A,group over dt (in place).
static __device__ __noinline__ void group_integrate(const EncParams& P, GroupState& g, double dt)
{
    const double h = dt / P.nsub;
    double kx[GMAX][3], kv[GMAX][3], tx[GMAX][3], tv[GMAX][3], ax[GMAX][3], av[GMAX][3];
    for (int s = 0; s < P.nsub; ++s) {
        group_rhs(P, g, g.x, g.v, kx, kv);
        for (int k = 0; k < g.n; ++k) for (int c = 0; c < 3; ++c) {
            ax[k][c] = kx[k][c]; av[k][c] = kv[k][c];
            tx[k][c] = fma(0.5 * h, kx[k][c], g.x[k][c]); tv[k][c] = fma(0.5 * h, kv[k][c], g.v[k][c]);
        }
        group_rhs(P, g, tx, tv, kx, kv);
        for (int k = 0; k < g.n; ++k) for (int c = 0; c < 3; ++c) {
            ax[k][c] += 2.0 * kx[k][c]; av[k][c] += 2.0 * kv[k][c];
            tx[k][c] = fma(0.5 * h, kx[k][c], g.x[k][c]); tv[k][c] = fma(0.5 * h, kv[k][c], g.v[k][c]);
        }
        group_rhs(P, g, tx, tv, kx, kv);
        for (int k = 0; k < g.n; ++k) for (int c = 0; c < 3; ++c) {
            ax[k][c] += 2.0 * kx[k][c]; av[k][c] += 2.0 * kv[k][c];
            tx[k][c] = fma(h, kx[k][c], g.x[k][c]); tv[k][c] = fma(h, kv[k][c], g.v[k][c]);
        }
        group_rhs(P, g, tx, tv, kx, kv);
        for (int k = 0; k < g.n; ++k) for (int c = 0; c < 3; ++c) {
            g.x[k][c] = fma(h / 6.0, ax[k][c] + kx[k][c], g.x[k][c]);
            g.v[k][c] = fma(h / 6.0, av[k][c] + kv[k][c], g.v[k][c]);
        }
    }
}

// The leader collects its group from the pair list (groups larger than GMAX were dissolved by group_kernel,
// fused_step.cu; the check here only guards the arrays).
__device__ __forceinline__ bool group_collect(int leader, const int2* __restrict__ pairs, unsigned int npairs,
                                              const int* __restrict__ glabel, GroupState& g, unsigned int* status)
{
    g.n = 1; g.body[0] = leader;
    for (unsigned int p = 0; p < npairs; ++p) {
        const int i = pairs[p].x, j = pairs[p].y;
        if (glabel[i] != leader) continue;
        for (int e = 0; e < 2; ++e) {
            const int b = e ? j : i;
            bool have = false;
            for (int k = 0; k < g.n; ++k) have = have || (g.body[k] == b);
            if (!have) {
                if (g.n == GMAX) { atomicOr(status, 2u); return false; }
                g.body[g.n++] = b;
            }
        }
    }
    return true;
}

}  // namespace enc
}  // namespace genga
