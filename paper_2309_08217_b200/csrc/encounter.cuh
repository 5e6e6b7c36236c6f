// encounter.cuh -- NEXT-1 (readings R11, R15), opt-in (params.encounter_mode = 1): the
// encounter complement of the hybrid symplectic step.  PAPER.md:45: "a changeover function smoothly switches"
// a pair between the fixed-step level-0 integrator and "the Bulirsch-Stoer integrator (level 1)"; PAPER.md:55,
// 159: close-encounter pairs and groups ("one big encounter group"); encounter forces always in
// double precision.
//
// During A(dt) a body that belongs to no encounter pair moves on its Kepler orbit (kepler.cuh).  The bodies of
// an encounter GROUP (a connected component of the pair list of the opening force evaluation) move under
//     H_A,group = sum_k (|p_k|^2 / 2 m_k - G M m_k / r_k) - sum_{k<l in group} G m_k m_l (1 - K(r_kl)) / r_kl,
// pair weight (1 - K) + r K' (the complement of the kick's K - r K'), r_crit,kl held at the values of the opening
// force evaluation (w.rcrit / w.semi / w.vkep / w.m, API order), all in FP64.
//
// A group is integrated by a TEAM with one thread per member: a warp for groups of up to WMAX = 16 bodies (the pair
// constants 1 / (0.9 r_crit,kl) in a table in shared memory), the whole CTA for groups of up to GBIG = 256 bodies
// (pair constants recomputed per pair: such groups are rare).  Members sit in ascending body index; a force
// evaluation writes the member's stage position to a double-buffered slab in shared memory, synchronises the team
// once and sums over the other members.  Integrators (the choice is params.enc_nsub):
//   * Gragg-Bulirsch-Stoer extrapolation to the relative tolerance params.enc_tol (default, reading R15): modified
//     midpoint with 2, 4, .. 16 substeps, polynomial extrapolation in h^2, error = largest |dx|/|x|, |dv|/|v| over
//     the members; a step that does not converge in 8 rows, or whose corrections stop falling (a pair crossing the
//     edge of its zone, where K is only C^1), is cut to a quarter; a step that converged in few rows is followed by
//     a longer one.  Status bit 8: the step size collapsed.  A warp team of up to 4 members runs the rows of the tableau
//     in parallel (integrate_bs_rows: lane = row x member, 2 r + 1 rounds of force evaluations for r rows instead of their
//     sum); teams of 3 to 6 members evaluate the ordered pairs of a force evaluation one per lane (accel).
//   * with params.enc_levels > 1 (reading R16): symplectic sub-levels with reduced steps between level 0 and the
//     Bulirsch-Stoer integration, which then only sees the innermost remainder of the pair potential.
//   * classical RK4 with enc_nsub equal substeps (the scheme of the first oracle, oracle_step_hybrid); with
//     params.enc_collide the members are tested for collisions after every substep and merged on the spot
//     (reading R14, oracle_step_hybrid_collide).
#pragma once

#include "genga_internal.cuh"

namespace genga {
namespace enc {

constexpr int WMAX = 16;           // largest group a warp integrates
constexpr int GBIG = 256;          // largest group at all: one CTA of the per-body kernel, one thread per member
constexpr int KMAX = 8;            // rows of the extrapolation tableau (substep counts 2, 4, .. 16)
constexpr unsigned int FULL = 0xffffffffu;

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

// 1/sqrt and 1/x from the MUFU seeds (rsqrt/rcp.approx.f64: about 2^-20 relative) with a cubic correction:
// relative error O(e^3) ~ 1e-18, i.e. a few ulp, at a fraction of the dependent latency of sqrt and divide.
__device__ __forceinline__ double rsq_seed(double a) { double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r; }
__device__ __forceinline__ double rcp_seed(double a) { double r; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r; }

// ---- shared memory of the teams ----------------------------------------------------------------------------------
struct WarpSlab {
    double pos[2][3][WMAX];        // stage positions of the members, double buffered
    double gm[WMAX], m[WMAX], rc[WMAX], sa[WMAX], vk[WMAX];   // rc < 0: the member was absorbed by a merger (reading R14)
    double i09[WMAX][WMAX];        // [l][k] = 1 / (0.9 r_crit,kl), 0: no zone (k == l, idle slots, absorbed members)
    double rad[WMAX], sum[8][WMAX];                          // collisions: radii, (m, m x, m v, R^3) of the members
    int    lab[WMAX], body[WMAX];
    __device__ __forceinline__ int body_of(int l) const { return body[l]; }
};
struct BlockSlab {
    double pos[2][3][GBIG];
    double gm[GBIG], m[GBIG], rc[GBIG], sa[GBIG], vk[GBIG];
    double rad[GBIG], sum[8][GBIG];
    double red[8];
    int    body[GBIG], lab[GBIG];
    __device__ __forceinline__ int body_of(int l) const { return body[l]; }
};
union EncSmem { WarpSlab w[8]; BlockSlab b; };     // warp teams and the CTA team never run at the same time

constexpr int PAIR_NMAX = 6;        // warp teams of up to this many members evaluate their pair terms one per lane (accel)

struct WarpTeam {
    static constexpr bool PAIR_LANES = true;            // the 32 lanes of the warp all call accel: idle ones can take pairs
    WarpSlab& s; int n, k;                              // k: member index of this lane, -1 for an idle lane
    int pi, pl;                                         // the ordered pair this lane evaluates in accel (member pl on member pi), -1: none
    __device__ __forceinline__ void sync() const { __syncwarp(); }
    __device__ __forceinline__ double maxall(double v) const
    {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(FULL, v, o));
        return v;
    }
    __device__ __forceinline__ double* px(int b) const { return s.pos[b][0]; }
    __device__ __forceinline__ double* py(int b) const { return s.pos[b][1]; }
    __device__ __forceinline__ double* pz(int b) const { return s.pos[b][2]; }
    __device__ __forceinline__ double gm(int l) const { return s.gm[l]; }
    __device__ __forceinline__ double inv09(const EncParams&, int l) const { return s.i09[l][k]; }
    // rebuild the pair table from the members' (possibly merged) masses; absorbed members have no zones
    __device__ __forceinline__ void refresh_pairs(const EncParams& P) const
    {
        __syncwarp();
        if (k >= 0)
            for (int l = 0; l < n; ++l) {
                const bool pair = (l != k) && s.rc[k] >= 0.0 && s.rc[l] >= 0.0;
                const double rc = pair ? pair_rcrit(P, s.m[k], s.m[l], s.rc[k], s.rc[l], s.sa[k], s.sa[l], s.vk[k], s.vk[l]) : 0.0;
                s.i09[l][k] = (rc > 0.0) ? 1.0 / (0.9 * rc) : 0.0;
            }
        __syncwarp();
    }
};
struct BlockTeam {
    static constexpr bool PAIR_LANES = false;
    BlockSlab& s; int n, k;
    __device__ __forceinline__ void sync() const { __syncthreads(); }
    __device__ __forceinline__ double maxall(double v) const
    {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(FULL, v, o));
        __syncthreads();                                   // red[] may still be read from the previous call
        if ((threadIdx.x & 31) == 0) s.red[threadIdx.x >> 5] = v;
        __syncthreads();
        double r = s.red[0];
#pragma unroll
        for (int q = 1; q < 8; ++q) r = fmax(r, s.red[q]);
        return r;
    }
    __device__ __forceinline__ double* px(int b) const { return s.pos[b][0]; }
    __device__ __forceinline__ double* py(int b) const { return s.pos[b][1]; }
    __device__ __forceinline__ double* pz(int b) const { return s.pos[b][2]; }
    __device__ __forceinline__ double gm(int l) const { return s.gm[l]; }
    __device__ __forceinline__ double inv09(const EncParams& P, int l) const
    {
        if (s.rc[k] < 0.0 || s.rc[l] < 0.0) return 0.0;     // absorbed by a merger
        const double rc = pair_rcrit(P, s.m[k], s.m[l], s.rc[k], s.rc[l], s.sa[k], s.sa[l], s.vk[k], s.vk[l]);
        return (rc > 0.0) ? 1.0 / (0.9 * rc) : 0.0;
    }
    __device__ __forceinline__ void refresh_pairs(const EncParams&) const { __syncthreads(); }   // recomputed per pair anyway
};

// ---- reading R14: collisions inside the encounter integration ("perfect mergers") ----------------------
// After a substep the members publish their positions; members k, l collide iff |x_k - x_l| < R_k + R_l (strict,
// plain sqrt as in oracle_merge).  Every connected component of that graph becomes one body at its smallest member
// (= smallest body index: members sit in ascending order): m = sum m, x = sum m x / m, v = sum m v / m,
// R = cbrt(sum R^3); a component of total mass 0 keeps its first member's x, v.  The absorbed members go on as
// massless bodies without zones (they exert and feel nothing but the star) until genga_merge closes the arrays up;
// absorb[body] names the body that took them.  Returns true if anything merged (uniform over the team).
template <class Team>
__device__ __forceinline__ bool collision_pass(const Team& T, const EncParams& P, int& buf, double (&y)[6], double& m,
                                               double& R, int body, int* __restrict__ absorb, Counters* ctr)
{
    double* X = T.px(buf); double* Y = T.py(buf); double* Z = T.pz(buf);
    const int k = T.k;
    const bool alive = k >= 0 && T.s.rc[k] >= 0.0;
    if (k >= 0) { X[k] = y[0]; Y[k] = y[1]; Z[k] = y[2]; T.s.rad[k] = alive ? R : -1.0; T.s.lab[k] = alive ? k : -1; }
    T.sync();
    buf ^= 1;
    auto touches = [&](int l) {
        if (l == k || T.s.rad[l] < 0.0) return false;
        const double dx = X[l] - y[0], dy = Y[l] - y[1], dz = Z[l] - y[2];
        return sqrt(dx * dx + dy * dy + dz * dz) < R + T.s.rad[l];
    };
    bool hit = false;
    if (alive) for (int l = 0; l < T.n; ++l) hit = hit || touches(l);
    if (!(T.maxall(hit ? 1.0 : 0.0) > 0.0)) return false;          // the usual substep
    // components by label propagation (labels = member indices)
    for (;;) {
        int lab = alive ? T.s.lab[k] : -1, nl = lab;
        if (alive) for (int l = 0; l < T.n; ++l) if (touches(l)) nl = min(nl, T.s.lab[l]);
        const bool changed = T.maxall(nl != lab ? 1.0 : 0.0) > 0.0;  // (team-wide sync inside for the CTA team)
        T.sync();
        if (alive) T.s.lab[k] = nl;
        T.sync();
        if (!changed) break;
    }
    if (k >= 0) {
        T.s.sum[0][k] = m; T.s.sum[1][k] = m * y[0]; T.s.sum[2][k] = m * y[1]; T.s.sum[3][k] = m * y[2];
        T.s.sum[4][k] = m * y[3]; T.s.sum[5][k] = m * y[4]; T.s.sum[6][k] = m * y[5]; T.s.sum[7][k] = R * R * R;
    }
    T.sync();
    if (alive) {
        const int root = T.s.lab[k];
        if (root == k) {
            int members = 0;
            double a[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            for (int l = k; l < T.n; ++l)
                if (T.s.lab[l] == k) { ++members; for (int c = 0; c < 8; ++c) a[c] += T.s.sum[c][l]; }
            if (members > 1) {
                if (a[0] > 0.0) { for (int c = 0; c < 3; ++c) { y[c] = a[1 + c] / a[0]; y[3 + c] = a[4 + c] / a[0]; } }
                m = a[0];
                R = cbrt(a[7]);
                atomicAdd(&ctr->enc_merged, (unsigned int)(members - 1));
            }
        } else {                                                    // absorbed by member `root`
            absorb[body] = T.s.body_of(root);
            m = 0.0; R = -1.0e300;                                  // never touches anything again
        }
    }
    T.sync();
    if (k >= 0) {
        const bool gone = alive && T.s.lab[k] != k;
        T.s.m[k] = m; T.s.gm[k] = P.G * m;
        if (gone) T.s.rc[k] = -1.0;
    }
    T.refresh_pairs(P);
    return true;
}

// W(q) = K - q K' for the zone of inverse width i09 = 1 / (0.9 r_crit) (readings G1, R10), branch-free: 0 below
// 0.1 r_crit, 1 from r_crit on.
__device__ __forceinline__ double zone_weight(double q, double i09)
{
    const double yy = fmin(fmax(fma(q, i09, -1.0 / 9.0), 0.0), 1.0);     // (q - 0.1 rc) / (0.9 rc)
    const double D  = fma(2.0 * yy, yy - 1.0, 1.0);                      // 2y^2 - 2y + 1, in [1/2, 1]
    const double r0 = rcp_seed(D), f = fma(-D, r0, 1.0);
    const double iD = fma(r0 * f, 1.0 + f, r0);
    const double K  = yy * yy * iD;
    const double Kp = 2.0 * yy * (1.0 - yy) * iD * iD * i09;             // dK/dr (0 at both ends)
    return K - q * Kp;
}

// dv/dt of this thread's member at the stage position (x, y, z): the member publishes its position in buffer buf,
// the team synchronises once, every member sums over the other members.  KEPLER: with the star's term -mu x / r^3.
// Pair weight: W(q; r_crit / fhi) - W(q; r_crit / flo), where fhi <= 0 stands for the constant 1: the complement of
// the two-level step is (flo, fhi) = (1, 0); shell l of the multi-level step (reading R16) is (F^(l-1), F^l), its
// innermost remainder (F^(L-1), 0).  Branch-free per pair.  Every thread of the team must call it.
template <bool KEPLER, class Team>
__device__ __forceinline__ void accel(const Team& T, const EncParams& P, int& buf, double x, double y, double z,
                                      double& a0, double& a1, double& a2, double flo = 1.0, double fhi = 0.0)
{
    double* X = T.px(buf); double* Y = T.py(buf); double* Z = T.pz(buf);
    if (T.k >= 0) { X[T.k] = x; Y[T.k] = y; Z[T.k] = z; }
    T.sync();
    buf ^= 1;                                              // the next evaluation writes the other buffer
    a0 = 0.0; a1 = 0.0; a2 = 0.0;
    if constexpr (Team::PAIR_LANES) {
        // A warp team of up to PAIR_NMAX members has a lane for every ORDERED pair (n (n - 1) <= 30): lane p takes the term of
        // member l on member i, i = p / (n - 1), and the member lanes collect theirs by shuffles.  The dependent chain of an
        // evaluation is then one pair (plus n - 1 shuffles) instead of n - 1 pairs: the drift waits for the slowest group.
        if (T.n >= 3 && T.n <= PAIR_NMAX) {                 // (a pair of bodies has nothing to gain)
            const int n1 = T.n - 1;
            const bool valid = T.pi >= 0;
            const int i = valid ? T.pi : 0, l = valid ? T.pl : 0;
            const double i09 = valid ? T.s.i09[l][i] : 0.0;
            const double d0 = X[l] - X[i], d1 = Y[l] - Y[i], d2 = Z[l] - Z[i];
            const double q2 = fma(d2, d2, fma(d1, d1, d0 * d0));
            const bool   on = (i09 > 0.0) && (q2 > 0.0);
            const double qs = on ? q2 : 1.0;
            const double y0 = rsq_seed(qs), t = y0 * y0, e = fma(-qs, t, 1.0), g = y0 * t;
            const double q0 = qs * y0;
            const double q  = fma(q0 * e, fma(0.375, e, 0.5), q0);              // |d|
            const double whi = (fhi > 0.0) ? zone_weight(q, i09 * fhi) : 1.0;
            const double Wc = on ? whi - zone_weight(q, i09 * flo) : 0.0;
            const double sc = T.gm(l) * Wc * fma(g * e, fma(1.875, e, 1.5), g);  // G m_l Wc / |d|^3
            const double c0 = sc * d0, c1 = sc * d1, c2 = sc * d2;
            if (KEPLER && T.k >= 0) {
                const double mu = P.G * P.M_star;
                const double r2 = fma(z, z, fma(y, y, x * x));
                const double u0 = rsq_seed(r2), tt = u0 * u0, ee = fma(-r2, tt, 1.0), gg = u0 * tt;
                const double ir3 = -mu * fma(gg * ee, fma(1.875, ee, 1.5), gg);  // -mu / r^3
                a0 = x * ir3; a1 = y * ir3; a2 = z * ir3;
            }
            const int base = (T.k >= 0) ? T.k * n1 : 0;
            for (int j = 0; j < n1; ++j) {
                const double v0 = __shfl_sync(FULL, c0, base + j), v1 = __shfl_sync(FULL, c1, base + j), v2 = __shfl_sync(FULL, c2, base + j);
                if (T.k >= 0) { a0 += v0; a1 += v1; a2 += v2; }
            }
            return;
        }
    }
    if (T.k < 0) return;
    if (KEPLER) {
        const double mu = P.G * P.M_star;
        const double r2 = fma(z, z, fma(y, y, x * x));
        const double y0 = rsq_seed(r2), t = y0 * y0, e = fma(-r2, t, 1.0), g = y0 * t;
        const double ir3 = -mu * fma(g * e, fma(1.875, e, 1.5), g);         // -mu / r^3
        a0 = x * ir3; a1 = y * ir3; a2 = z * ir3;
    }
    // the other members, starting with the next one (member k takes l = k + 1, k + 2, .. cyclically): a pair costs
    // one pass of this dependent chain, which is what the drift's duration is made of
#pragma unroll 2
    for (int j = 1; j < T.n; ++j) {
        const int l = (T.k + j < T.n) ? T.k + j : T.k + j - T.n;
        const double i09 = T.inv09(P, l);
        const double d0 = X[l] - x, d1 = Y[l] - y, d2 = Z[l] - z;
        const double q2 = fma(d2, d2, fma(d1, d1, d0 * d0));
        const bool   on = (i09 > 0.0) && (q2 > 0.0);
        const double qs = on ? q2 : 1.0;
        const double y0 = rsq_seed(qs), t = y0 * y0, e = fma(-qs, t, 1.0), g = y0 * t;
        const double q0 = qs * y0;
        const double q  = fma(q0 * e, fma(0.375, e, 0.5), q0);              // |d|
        const double whi = (fhi > 0.0) ? zone_weight(q, i09 * fhi) : 1.0;
        const double Wc = on ? whi - zone_weight(q, i09 * flo) : 0.0;
        const double s  = T.gm(l) * Wc * fma(g * e, fma(1.875, e, 1.5), g);  // G m_l Wc / |d|^3
        a0 = fma(s, d0, a0); a1 = fma(s, d1, a1); a2 = fma(s, d2, a2);
    }
}

// P.collide: after every substep the collision pass of reading R14 (m, R: this member's mass and radius, updated).
template <bool COLL, class Team>
__device__ __forceinline__ void integrate_rk4(const Team& T, const EncParams& P, double dt, double (&y)[6], Counters* ctr,
                                              double& m, double& R, int body, int* __restrict__ absorb)
{
    const double h = dt / P.nsub, hh = 0.5 * h, h6 = h / 6.0;
    int buf = 0;
    for (int s = 0; s < P.nsub; ++s) {
        double k0, k1, k2, sx[3], sv[3], t[3], u[3];
        accel<true>(T, P, buf, y[0], y[1], y[2], k0, k1, k2);
        sx[0] = y[3]; sx[1] = y[4]; sx[2] = y[5]; sv[0] = k0; sv[1] = k1; sv[2] = k2;
        t[0] = fma(hh, y[3], y[0]); t[1] = fma(hh, y[4], y[1]); t[2] = fma(hh, y[5], y[2]);
        u[0] = fma(hh, k0, y[3]); u[1] = fma(hh, k1, y[4]); u[2] = fma(hh, k2, y[5]);
        accel<true>(T, P, buf, t[0], t[1], t[2], k0, k1, k2);
        sx[0] += 2.0 * u[0]; sx[1] += 2.0 * u[1]; sx[2] += 2.0 * u[2]; sv[0] += 2.0 * k0; sv[1] += 2.0 * k1; sv[2] += 2.0 * k2;
        t[0] = fma(hh, u[0], y[0]); t[1] = fma(hh, u[1], y[1]); t[2] = fma(hh, u[2], y[2]);
        u[0] = fma(hh, k0, y[3]); u[1] = fma(hh, k1, y[4]); u[2] = fma(hh, k2, y[5]);
        accel<true>(T, P, buf, t[0], t[1], t[2], k0, k1, k2);
        sx[0] += 2.0 * u[0]; sx[1] += 2.0 * u[1]; sx[2] += 2.0 * u[2]; sv[0] += 2.0 * k0; sv[1] += 2.0 * k1; sv[2] += 2.0 * k2;
        t[0] = fma(h, u[0], y[0]); t[1] = fma(h, u[1], y[1]); t[2] = fma(h, u[2], y[2]);
        u[0] = fma(h, k0, y[3]); u[1] = fma(h, k1, y[4]); u[2] = fma(h, k2, y[5]);
        accel<true>(T, P, buf, t[0], t[1], t[2], k0, k1, k2);
        y[0] = fma(h6, sx[0] + u[0], y[0]); y[1] = fma(h6, sx[1] + u[1], y[1]); y[2] = fma(h6, sx[2] + u[2], y[2]);
        y[3] = fma(h6, sv[0] + k0, y[3]); y[4] = fma(h6, sv[1] + k1, y[4]); y[5] = fma(h6, sv[2] + k2, y[5]);
        if (COLL && P.collide) collision_pass(T, P, buf, y, m, R, body, absorb, ctr);
    }
    if (T.k == 0) { atomicAdd(&ctr->enc_rhs_sum, 4u * (unsigned int)P.nsub); atomicMax(&ctr->enc_rhs_max, 4u * (unsigned int)P.nsub); }
}

// Gragg-Bulirsch-Stoer for a warp team of up to ROWS_NMAX members with the rows of the extrapolation tableau IN PARALLEL:
// the rows (2, 4, .. 16 modified-midpoint substeps over the same macro step H) do not depend on one another, and a warp that
// integrates a pair of bodies has 30 idle lanes.  Lane r n + k carries member k through row r (n_r = 2 (r + 1) substeps);
// the members of a row see each other's stage positions by shuffles (no shared-memory slab, no barrier).  A macro step
// with r rows costs 2 r + 1 rounds of force evaluations (17 for all eight), against 3 + 5 + .. (2 k + 3) = 24, 35, 48 rounds
// when the rows run one after the other and row k = 3, 4, 5 converges, and 80 for a rejected step.  Measured: ~1100 cycles per
// round for a team of three, of which ~300 are the macro step's own (first evaluation, tableau, decisions).  Same arithmetic per row, same
// acceptance and step-size rules as integrate_bs; the tableau is spread over the lanes as well (no arrays in local memory, no
// divisions per macro step), which changes its rounding, not its values.
// Every lane keeps the state of ITS member (y, replicated over the rows).  Must be called by the whole warp, converged.
constexpr int ROWS_NMAX = 32 / KMAX;

// Complement weight 1 - W(q; zone of inverse width i09) = 1 - K + q K' with one reciprocal: K = u^2 / D, K' = 2 u (1 - u) i09 / D^2,
// u = clamp((q - 0.1 rc) / (0.9 rc)), D = 2 u^2 - 2 u + 1  =>  1 - W = (D^2 - u^2 D + 2 q i09 u (1 - u)) / D^2.  (zone_weight() forms
// K and K' one after the other; the two agree to rounding.  Shorter dependent chain: this is what a round waits for.)
__device__ __forceinline__ double zone_complement(double q, double i09)
{
    const double u  = fmin(fmax(fma(q, i09, -1.0 / 9.0), 0.0), 1.0);
    const double D  = fma(2.0 * u, u - 1.0, 1.0), D2 = D * D;
    const double r0 = rcp_seed(D2), f = fma(-D2, r0, 1.0);
    const double iD2 = fma(r0 * f, 1.0 + f, r0);
    const double num = fma(2.0 * q * i09, u * (1.0 - u), fma(-u * u, D, D2));
    return num * iD2;
}

// Force evaluation of the row-parallel integrator for a team of N members, fully unrolled: the N - 1 pair terms of a
// lane are independent chains that overlap.  gmo / i09o: G m and 1 / (0.9 r_crit / flo) of the other members, in the
// order l = mem + 1, mem + 2, .. (cyclic), held in registers for the whole integration.
template <int N>
__device__ __forceinline__ void rows_accel(double mu, int rbase, int mem, const double (&gmo)[N > 1 ? N - 1 : 1],
                                           const double (&i09o)[N > 1 ? N - 1 : 1], double x, double y, double z,
                                           double& a0, double& a1, double& a2)
{
    // All shuffles first: a shuffle is a barrier for the compiler's scheduling, and with one per pair in front of its
    // arithmetic the pair chains (and the star's) ran one after the other (measured: +370 cycles per member).
    double xl[N > 1 ? N - 1 : 1], yl[N > 1 ? N - 1 : 1], zl[N > 1 ? N - 1 : 1];
#pragma unroll
    for (int j = 1; j < N; ++j) {                                               // the other members, in the order of accel()
        const int l = (mem + j < N) ? mem + j : mem + j - N;
        xl[j - 1] = __shfl_sync(FULL, x, rbase + l); yl[j - 1] = __shfl_sync(FULL, y, rbase + l); zl[j - 1] = __shfl_sync(FULL, z, rbase + l);
    }
    const double r2 = fma(z, z, fma(y, y, x * x));
    const double u0 = rsq_seed(r2), tt = u0 * u0, ee = fma(-r2, tt, 1.0), gg = u0 * tt;
    const double ir3 = -mu * fma(gg * ee, fma(1.875, ee, 1.5), gg);             // -mu / r^3
    a0 = x * ir3; a1 = y * ir3; a2 = z * ir3;
    double s0[N > 1 ? N - 1 : 1], s1[N > 1 ? N - 1 : 1], s2[N > 1 ? N - 1 : 1];
#pragma unroll
    for (int j = 1; j < N; ++j) {
        const double i09 = i09o[j - 1];
        const double d0 = xl[j - 1] - x, d1 = yl[j - 1] - y, d2 = zl[j - 1] - z;
        const double q2 = fma(d2, d2, fma(d1, d1, d0 * d0));
        const bool   on = (i09 > 0.0) && (q2 > 0.0);
        const double qs = on ? q2 : 1.0;
        const double y0 = rsq_seed(qs), t = y0 * y0, e = fma(-qs, t, 1.0), g = y0 * t;
        const double q0 = qs * y0;
        const double q  = fma(q0 * e, fma(0.375, e, 0.5), q0);                  // |d|
        const double Wc = on ? zone_complement(q, i09) : 0.0;
        const double sc = gmo[j - 1] * Wc * fma(g * e, fma(1.875, e, 1.5), g);   // G m_l Wc / |d|^3
        s0[j - 1] = sc * d0; s1[j - 1] = sc * d1; s2[j - 1] = sc * d2;
    }
#pragma unroll
    for (int j = 1; j < N; ++j) { a0 += s0[j - 1]; a1 += s1[j - 1]; a2 += s2[j - 1]; }   // summed in the order of accel()
}

template <int N>
__device__ __forceinline__ void integrate_bs_rows(const WarpTeam& T, const EncParams& P, double dt, double (&y)[6], Counters* ctr,
                                                  double flo)
{
    constexpr int n = N;
    const int lane = threadIdx.x & 31;
    const bool act = lane < KMAX * n;
    const int row = act ? lane / n : 0, mem = act ? lane - row * n : 0, rbase = row * n;
    const int nk = 2 * (row + 1);
    // every lane takes over the state of its member
#pragma unroll
    for (int c = 0; c < 6; ++c) y[c] = __shfl_sync(FULL, y[c], mem);
    const double mu = P.G * P.M_star;
    double gmo[N - 1], i09o[N - 1];
#pragma unroll
    for (int j = 1; j < N; ++j) {
        const int l = (mem + j < N) ? mem + j : mem + j - N;
        gmo[j - 1] = T.gm(l); i09o[j - 1] = T.s.i09[l][mem] * flo;
    }
    // Aitken-Neville in h^2 with the tableau spread over the lanes: lane (r, k) holds T[r][j] of its member, column after
    // column, and takes T[r-1][j-1] from the lane n below: T[r][j] = T[r][j-1] + (T[r][j-1] - T[r-1][j-1]) / ((n_r / n_(r-j))^2 - 1).
    // (The sequential form keeps the same tableau as differences in an array; the two agree to rounding.)
    double cj[KMAX];
#pragma unroll
    for (int j = 1; j < KMAX; ++j) {
        const double q = (j <= row) ? (double)(row + 1) / (double)(row + 1 - j) : 2.0;
        cj[j] = 1.0 / (q * q - 1.0);
    }
    const double Tabs = fabs(dt);
    double t = 0.0, H = dt;
    bool collapsed = false;
    unsigned int nrhs = 0u, nrej = 0u;
    // Rows actually run: two beyond the row that converged last time (17 rounds for all eight would be more than the
    // sequential form needs when row 2 or 3 converges); if they do not settle the step, it is redone with all eight.  The
    // decisions are taken row by row in the same order either way, so the result does not depend on this guess.
    int rows_use = KMAX;
    while (fabs(t) < Tabs * (1.0 - 1.0e-14)) {
        if (fabs(t + H) > Tabs) H = dt - t;
        double f0[3];
        rows_accel<N>(mu, rbase, mem, gmo, i09o, y[0], y[1], y[2], f0[0], f0[1], f0[2]);
        ++nrhs;
        const double h = H / nk, h2 = 2.0 * h;
        double z0[6], z1[6], f[3], est[6];
        int done = -1;
        for (int ru = rows_use;;) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { z0[c] = y[c]; z0[3 + c] = y[3 + c]; z1[c] = fma(h, y[3 + c], y[c]); z1[3 + c] = fma(h, f0[c], y[3 + c]); }
#pragma unroll
        for (int c = 0; c < 6; ++c) est[c] = 0.0;
        for (int s = 1; s <= 2 * ru; ++s) {                                      // round s: the rows with n_r >= s are still under way
            rows_accel<N>(mu, rbase, mem, gmo, i09o, z1[0], z1[1], z1[2], f[0], f[1], f[2]);
            // (by selection, not by branches: the rows of a warp are at different places of their midpoint rules)
            const bool step = s < nk, fin = s == nk;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double nx = fma(h2, z1[3 + c], z0[c]), nv = fma(h2, f[c], z0[3 + c]);
                const double ex = 0.5 * (z1[c] + z0[c] + h * z1[3 + c]), ev = 0.5 * (z1[3 + c] + z0[3 + c] + h * f[c]);
                est[c] = fin ? ex : est[c]; est[3 + c] = fin ? ev : est[3 + c];
                z0[c] = step ? z1[c] : z0[c]; z0[3 + c] = step ? z1[3 + c] : z0[3 + c];
                z1[c] = step ? nx : z1[c]; z1[3 + c] = step ? nv : z1[3 + c];
            }
        }
        nrhs += 2u * (unsigned int)ru;
        // the tableau (see above): after column j the lanes of row r >= j hold T[r][j]; last = T[r][r] - T[r][r-1]
        double last[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int j = 1; j < KMAX; ++j) {
            if (j < ru) {
                double prev[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) prev[c] = __shfl_sync(FULL, est[c], (lane >= n) ? lane - n : lane);
                if (act && row >= j && row < ru) {
#pragma unroll
                    for (int c = 0; c < 6; ++c) {
                        const double corr = (est[c] - prev[c]) * cj[j];
                        est[c] += corr;
                        if (j == row) last[c] = corr;
                    }
                }
            }
        }
        // error of row r: its last correction against its value, the largest over the members of the row
        double e = 0.0;
        if (act && row >= 1 && row < ru) {
            const double ex = (last[0] * last[0] + last[1] * last[1] + last[2] * last[2]) / (est[0] * est[0] + est[1] * est[1] + est[2] * est[2]);
            const double ev = (last[3] * last[3] + last[4] * last[4] + last[5] * last[5]) / (est[3] * est[3] + est[4] * est[4] + est[5] * est[5]);
            e = fmax(ex, ev);
            if (!(e == e)) e = 1.0e300;                   // NaN: not converged
        }
        {
            double em = e;
            for (int l = 0; l < n; ++l) em = fmax(em, __shfl_sync(FULL, e, rbase + l));
            e = em;
        }
        // the decisions, row by row in the order of the sequential form
        double eprev = 1.0e300;
        bool stalled = false;
        done = -1;
        for (int k = 1; k < ru; ++k) {
            const double ek = __shfl_sync(FULL, e, k * n);
            if (ek <= P.tol * P.tol) { done = k; break; }
            if (k >= 3 && ek > 0.04 * eprev) { stalled = true; break; }   // the corrections stopped falling: a zone edge inside the step
            eprev = ek;
        }
        if (done >= 0 || stalled || ru == KMAX) break;
        ru = KMAX;                                                               // not settled by the rows run: all eight
        }
        if (done < 0) {
            ++nrej;
            H *= 0.25;
            rows_use = 6;
            if (fabs(H) < Tabs * 9.3e-10) { collapsed = true; break; }
            continue;
        }
        rows_use = min(KMAX, max(3, done + 2));
#pragma unroll
        for (int c = 0; c < 6; ++c) y[c] = __shfl_sync(FULL, est[c], done * n + mem);
        t += H;
        H = (done <= 2) ? 4.0 * H : ((done <= 4) ? 2.0 * H : ((done <= 5) ? H : 0.5 * H));
    }
    if (lane == 0) {
        if (collapsed) atomicOr(&ctr->enc_status, 8u);
        atomicAdd(&ctr->enc_rhs_sum, nrhs); atomicMax(&ctr->enc_rhs_max, nrhs); atomicAdd(&ctr->enc_rejected, nrej);
    }
}


// A(dt) by Gragg-Bulirsch-Stoer extrapolation to the relative tolerance P.tol (reading R15).  The tableau is kept in
// the difference form of polynomial extrapolation (one column of differences per row), which yields the extrapolated
// value and the last correction, i.e. the error estimate T_kk - T_k,k-1, without storing two rows.
template <class Team>
__device__ __forceinline__ void integrate_bs(const Team& T, const EncParams& P, double dt, double (&y)[6], Counters* ctr,
                                             double flo = 1.0)
{
    if constexpr (Team::PAIR_LANES) {
        // the rows of the tableau in parallel
        if (T.n == 2) { integrate_bs_rows<2>(T, P, dt, y, ctr, flo); return; }
        if (T.n == 3) { integrate_bs_rows<3>(T, P, dt, y, ctr, flo); return; }
        if (T.n == 4) { integrate_bs_rows<4>(T, P, dt, y, ctr, flo); return; }
        static_assert(ROWS_NMAX == 4, "one instance per team size");
    }
    const double Tabs = fabs(dt);
    double t = 0.0, H = dt;
    int buf = 0;
    bool collapsed = false;
    unsigned int nrhs = 0u, nrej = 0u;
    while (fabs(t) < Tabs * (1.0 - 1.0e-14)) {
        if (fabs(t + H) > Tabs) H = dt - t;
        double f0[3];
        accel<true>(T, P, buf, y[0], y[1], y[2], f0[0], f0[1], f0[2], flo);
        ++nrhs;
        double d[KMAX][6], hsq[KMAX], yz[6], dy[6];
        double eprev = 1.0e300;
        int done = -1;
        for (int k = 0; k < KMAX && done < 0; ++k) {
            const int nk = 2 * (k + 1);
            const double h = H / nk, h2 = 2.0 * h;
            double z0[6], z1[6], f[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) { z0[c] = y[c]; z0[3 + c] = y[3 + c]; z1[c] = fma(h, y[3 + c], y[c]); z1[3 + c] = fma(h, f0[c], y[3 + c]); }
            for (int s = 1; s < nk; ++s) {
                accel<true>(T, P, buf, z1[0], z1[1], z1[2], f[0], f[1], f[2], flo);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const double nx = fma(h2, z1[3 + c], z0[c]), nv = fma(h2, f[c], z0[3 + c]);
                    z0[c] = z1[c]; z0[3 + c] = z1[3 + c]; z1[c] = nx; z1[3 + c] = nv;
                }
            }
            accel<true>(T, P, buf, z1[0], z1[1], z1[2], f[0], f[1], f[2], flo);
            nrhs += (unsigned int)nk;
            double est[6];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                est[c] = 0.5 * (z1[c] + z0[c] + h * z1[3 + c]);
                est[3 + c] = 0.5 * (z1[3 + c] + z0[3 + c] + h * f[c]);
            }
            // polynomial extrapolation to h^2 = 0 through the rows 0 .. k
            hsq[k] = h * h;
#pragma unroll
            for (int c = 0; c < 6; ++c) { yz[c] = est[c]; dy[c] = est[c]; }
            if (k == 0) {
#pragma unroll
                for (int c = 0; c < 6; ++c) d[0][c] = est[c];
            } else {
                double cc[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) cc[c] = est[c];
                for (int j = 0; j < k; ++j) {
                    const double delta = 1.0 / (hsq[k - j - 1] - hsq[k]);
                    const double f1 = hsq[k] * delta, f2 = hsq[k - j - 1] * delta;
#pragma unroll
                    for (int c = 0; c < 6; ++c) {
                        const double q = d[j][c];
                        d[j][c] = dy[c];
                        const double dl = cc[c] - q;
                        dy[c] = f1 * dl; cc[c] = f2 * dl;
                        yz[c] += dy[c];
                    }
                }
#pragma unroll
                for (int c = 0; c < 6; ++c) d[k][c] = dy[c];
                double e = 0.0;
                if (T.k >= 0) {
                    const double ex = (dy[0] * dy[0] + dy[1] * dy[1] + dy[2] * dy[2]) / (yz[0] * yz[0] + yz[1] * yz[1] + yz[2] * yz[2]);
                    const double ev = (dy[3] * dy[3] + dy[4] * dy[4] + dy[5] * dy[5]) / (yz[3] * yz[3] + yz[4] * yz[4] + yz[5] * yz[5]);
                    e = fmax(ex, ev);
                    if (!(e == e)) e = 1.0e300;           // NaN: not converged
                }
                e = T.maxall(e);
                if (e <= P.tol * P.tol) done = k;         // squared norms against the squared tolerance
                // A pair that crosses the edge of its zone inside the step (K is C^1 there) makes the corrections
                // stagnate instead of falling row by row: give the step up early rather than after all 8 rows.
                else if (k >= 3 && e > 0.04 * eprev) k = KMAX;
                eprev = e;
            }
        }
        if (done < 0) {
            ++nrej;
            H *= 0.25;
            if (fabs(H) < Tabs * 9.3e-10) { collapsed = true; break; }      // dt 2^-30: give up, keep the last accepted state
            continue;
        }
#pragma unroll
        for (int c = 0; c < 6; ++c) y[c] = yz[c];
        t += H;
        H = (done <= 2) ? 4.0 * H : ((done <= 4) ? 2.0 * H : ((done <= 5) ? H : 0.5 * H));
    }
    if (T.k == 0) {
        if (collapsed) atomicOr(&ctr->enc_status, 8u);
        atomicAdd(&ctr->enc_rhs_sum, nrhs); atomicMax(&ctr->enc_rhs_max, nrhs); atomicAdd(&ctr->enc_rejected, nrej);
    }
}

// Reading R16: flow_l(tau) of H_Kep + (1 - W_{l-1}) V for the group.  l == levels: Bulirsch-Stoer
// with the innermost remainder; otherwise levels_sub times [ kick_l(h/2) flow_{l+1}(h) kick_l(h/2) ], h = tau / sub,
// kick_l: v += (h/2) a with the shell weight W_l - W_{l-1} (radius ratio F per level).  fl = F^(l-1).
constexpr int LMAX = 4;            // most changeover levels (no recursion on the device: the levels are unrolled)

template <class Team>
__device__ __noinline__ void bs_call(const Team& T, const EncParams& P, double tau, double (&y)[6], Counters* ctr, double fl)
{
    integrate_bs(T, P, tau, y, ctr, fl);
}

template <int LVL, class Team>
__device__ __forceinline__ void level_flow(const Team& T, const EncParams& P, double fl, double tau, double (&y)[6], Counters* ctr)
{
    if constexpr (LVL >= LMAX) {
        bs_call(T, P, tau, y, ctr, fl);
    } else {
        if (LVL >= P.levels) { bs_call(T, P, tau, y, ctr, fl); return; }
        const double h = tau / P.levels_sub, hh = 0.5 * h, fh = fl * P.level_ratio;
        int buf = 0;
        for (int s = 0; s < P.levels_sub; ++s) {
            double a0, a1, a2;
            accel<false>(T, P, buf, y[0], y[1], y[2], a0, a1, a2, fl, fh);
            y[3] = fma(hh, a0, y[3]); y[4] = fma(hh, a1, y[4]); y[5] = fma(hh, a2, y[5]);
            T.sync();                                       // the slab buffers are reused by the inner level
            level_flow<LVL + 1>(T, P, fh, h, y, ctr);
            T.sync();
            accel<false>(T, P, buf, y[0], y[1], y[2], a0, a1, a2, fl, fh);
            y[3] = fma(hh, a0, y[3]); y[4] = fma(hh, a1, y[4]); y[5] = fma(hh, a2, y[5]);
        }
    }
}

// FULL: with the in-drift collisions (reading R14) and the sub-levels (reading R16).  The per-body kernel is compiled
// twice: the plain instance (Bulirsch-Stoer or RK4 of the two-level step) keeps its registers; the full one spills.
template <bool FULL_FEATURES, class Team>
__device__ __forceinline__ void integrate(const Team& T, const EncParams& P, double dt, double (&y)[6], Counters* ctr,
                                          double& m, double& R, int body, int* __restrict__ absorb)
{
    if (dt == 0.0) return;
    if (P.nsub > 0)                         integrate_rk4<FULL_FEATURES>(T, P, dt, y, ctr, m, R, body, absorb);
    else if (FULL_FEATURES && P.levels > 1) level_flow<1>(T, P, 1.0, dt, y, ctr);
    else                                    integrate_bs(T, P, dt, y, ctr);
}

// Groups in Workspace::ginfo (written by group_kernel): ginfo[2 g] = offset of the member list, ginfo[2 g + 1] = member
// count; the member lists (body indices, in no particular order) follow from ginfo[2 maxgroups] on.
__device__ __forceinline__ const int* group_members(const Workspace& w, int maxgroups, int g, int& n)
{
    n = w.ginfo[2 * g + 1];
    return w.ginfo + 2 * (size_t)maxgroups + w.ginfo[2 * g];
}

// One warp advances a group of n <= WMAX bodies through S(dt/2) (the shift s, already scaled) and the flow of
// H_A,group over dt, and writes its members back.  Members are taken in ascending body index, so the result does
// not depend on the order in which group_kernel registered them.
template <bool FULL_FEATURES>
__device__ __forceinline__ void warp_group(const EncParams& P, Workspace& w, WarpSlab& slab, const int* mem, int n,
                                           double dt, double s0, double s1, double s2)
{
    const int lane = threadIdx.x & 31;
    const int b_in = (lane < n) ? mem[lane] : 0x7fffffff;
    int rank = 0;
    for (int l = 0; l < n; ++l) { const int o = __shfl_sync(FULL, b_in, l); if (o < b_in) ++rank; }
    int b = -1;
    for (int l = 0; l < n; ++l) {
        const int o = __shfl_sync(FULL, b_in, l), r = __shfl_sync(FULL, rank, l);
        if (r == lane) b = o;
    }
    const bool active = lane < n;
    double m = 0.0, rci = 0.0, sa = 0.0, vk = 0.0;
    double y[6] = {1.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    if (active) {
        m = w.m[b]; rci = w.rcrit[b]; sa = w.semi[b]; vk = w.vkep[b];
        y[0] = w.x[3 * b] + s0; y[1] = w.x[3 * b + 1] + s1; y[2] = w.x[3 * b + 2] + s2;
        y[3] = w.v[3 * b]; y[4] = w.v[3 * b + 1]; y[5] = w.v[3 * b + 2];
    }
    __syncwarp();                                           // the slab may still be read by the previous group's last sum
    double R = 0.0;
    if (active) {
        slab.m[lane] = m; slab.gm[lane] = P.G * m; slab.rc[lane] = rci; slab.sa[lane] = sa; slab.vk[lane] = vk; slab.body[lane] = b;
        if (P.collide) R = w.radius[b];
    }
    int pi = -1, pl = -1;
    if (n >= 3 && n <= PAIR_NMAX && lane < n * (n - 1)) { pi = lane / (n - 1); const int jj = lane - pi * (n - 1); pl = jj + (jj >= pi ? 1 : 0); }
    const WarpTeam T{slab, n, active ? lane : -1, pi, pl};
    T.refresh_pairs(P);
    integrate<FULL_FEATURES>(T, P, dt, y, w.ctr, m, R, b, w.absorb);
    if (active) {
        w.x[3 * b] = y[0]; w.x[3 * b + 1] = y[1]; w.x[3 * b + 2] = y[2];
        w.v[3 * b] = y[3]; w.v[3 * b + 1] = y[4]; w.v[3 * b + 2] = y[5];
        if (P.collide) { w.m[b] = m; w.radius[b] = R; w.hcbrt[b] = cbrt(m / (3.0 * P.M_star)); }
    }
}

// The whole CTA (GBIG threads) advances a group of WMAX < n <= GBIG bodies.  Must be called by all threads.
template <bool FULL_FEATURES>
__device__ __forceinline__ void block_group(const EncParams& P, Workspace& w, BlockSlab& slab, const int* mem, int n,
                                            double dt, double s0, double s1, double s2)
{
    const int tid = threadIdx.x;
    __syncthreads();                                        // the slab (a union with the warp slabs) is free
    const int b_in = (tid < n) ? mem[tid] : 0x7fffffff;
    if (tid < n) slab.body[tid] = b_in;
    __syncthreads();
    int rank = 0;
    if (tid < n) for (int l = 0; l < n; ++l) if (slab.body[l] < b_in) ++rank;
    __syncthreads();
    if (tid < n) slab.body[rank] = b_in;                    // ascending body index (indices are distinct)
    __syncthreads();
    const bool active = tid < n;
    double y[6] = {1.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    double mm = 0.0, R = 0.0;
    int b = -1;
    if (active) {
        b = slab.body[tid];
        const double m = w.m[b];
        slab.m[tid] = m; slab.gm[tid] = P.G * m; slab.rc[tid] = w.rcrit[b]; slab.sa[tid] = w.semi[b]; slab.vk[tid] = w.vkep[b];
        mm = m;
        if (P.collide) R = w.radius[b];
        y[0] = w.x[3 * b] + s0; y[1] = w.x[3 * b + 1] + s1; y[2] = w.x[3 * b + 2] + s2;
        y[3] = w.v[3 * b]; y[4] = w.v[3 * b + 1]; y[5] = w.v[3 * b + 2];
    }
    __syncthreads();
    const BlockTeam T{slab, n, active ? tid : -1};
    integrate<FULL_FEATURES>(T, P, dt, y, w.ctr, mm, R, b, w.absorb);
    if (active) {
        w.x[3 * b] = y[0]; w.x[3 * b + 1] = y[1]; w.x[3 * b + 2] = y[2];
        w.v[3 * b] = y[3]; w.v[3 * b + 1] = y[4]; w.v[3 * b + 2] = y[5];
        if (P.collide) { w.m[b] = mm; w.radius[b] = R; w.hcbrt[b] = cbrt(mm / (3.0 * P.M_star)); }
    }
    __syncthreads();
}

}  // namespace enc
}  // namespace genga
