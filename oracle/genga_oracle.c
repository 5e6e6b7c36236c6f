/*
 * genga_oracle.c -- CPU FP64 oracle for the GENGA level-0 hot path (see genga_oracle.h).
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Plain C99, FP64, sqrt + divide, j ascending,
 * Neumaier-compensated sums; OpenMP over i only (each body's own sum has a fixed order, so
 * results do not depend on the thread count).  No code is shared with the CUDA path.
 *
 * Citations: PAPER.md:NN = line NN of /root/reference/PAPER.md.  O1..O11 and G1..G11 are
 * the oracle steps and readings of SURVEY.md section 8(c), restated in DESIGN.md section 3.
 *
 * Build:  gcc -std=c99 -O2 -ffp-contract=off -fopenmp -fPIC -shared genga_oracle.c -lm
 */
#include "genga_oracle.h"

#include <math.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- Neumaier compensated accumulator: value = s + c ------------------------------------ */
typedef struct { double s, c; } nsum;

static void nsum_add(nsum* a, double t)
{
    double S = a->s + t;
    if (fabs(a->s) >= fabs(t)) a->c += (a->s - S) + t;
    else                       a->c += (t - S) + a->s;
    a->s = S;
}
static double nsum_value(const nsum* a) { return a->s + a->c; }

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- O4: changeover function, reading G1 ---------------------------------------------------
 * PAPER.md:45 "A changeover function smoothly switches between the two levels (Chambers
 * 1999)".  The formula is not printed; reading G1 takes the rational form
 *   y = (r - 0.1 rc)/(0.9 rc);  K = 0 (y <= 0),  y^2/(2y^2 - 2y + 1) (0 < y < 1),  1 (y >= 1).
 * rc <= 0 means "no changeover zone": K = 1 for every r > 0.                                  */
double oracle_changeover(double r, double rcrit)
{
    if (!(rcrit > 0.0)) return (r > 0.0) ? 1.0 : 0.0;
    double y = (r - 0.1 * rcrit) / (0.9 * rcrit);
    if (y <= 0.0) return 0.0;
    if (y >= 1.0) return 1.0;
    return (y * y) / (2.0 * y * y - 2.0 * y + 1.0);
}

/* Pair weight (reading G1b / R10).  mode 0: W = K (north_star: "weighted by the changeover function
 * K").  mode 1: W = K - r dK/dr, the weight that makes the kick the gradient of the K-weighted pair
 * potential -G m_i m_j K(r)/r:  -d/dr [K/r] = (K - r K')/r^2.  With y = (r - 0.1 rc)/(0.9 rc) and
 * K = y^2/D, D = 2y^2 - 2y + 1:  dK/dy = 2y(1 - y)/D^2, dK/dr = dK/dy / (0.9 rc); K' = 0 outside 0<y<1. */
double oracle_weight(double r, double rcrit, int mode)
{
    double K = oracle_changeover(r, rcrit);
    if (mode == 0 || !(rcrit > 0.0)) return K;
    double y = (r - 0.1 * rcrit) / (0.9 * rcrit);
    if (y <= 0.0 || y >= 1.0) return K;
    double D = 2.0 * y * y - 2.0 * y + 1.0;
    double dKdr = (2.0 * y * (1.0 - y) / (D * D)) / (0.9 * rcrit);
    return K - r * dKdr;
}

/* ---- O1: velocity conventions, reading G3 -------------------------------------------------
 * stored v_i = v_h,i - (sum_j m_j v_h,j)/(M_star + sum_j m_j);
 * inverse    v_h,i = v_i + (sum_j m_j v_j)/M_star.                                            */
static void mass_weighted_velocity(int N, const double* m, const double* v, double out[3], double* mtot)
{
    nsum p[3] = {{0, 0}, {0, 0}, {0, 0}}, mt = {0, 0};
    for (int j = 0; j < N; ++j) {
        for (int k = 0; k < 3; ++k) nsum_add(&p[k], m[j] * v[3 * j + k]);
        nsum_add(&mt, m[j]);
    }
    for (int k = 0; k < 3; ++k) out[k] = nsum_value(&p[k]);
    if (mtot) *mtot = nsum_value(&mt);
}

void oracle_to_democratic(int N, const double* m, double* v, double M_star)
{
    double p[3], mt;
    mass_weighted_velocity(N, m, v, p, &mt);
    for (int i = 0; i < N; ++i)
        for (int k = 0; k < 3; ++k) v[3 * i + k] -= p[k] / (M_star + mt);
}

void oracle_to_heliocentric(int N, const double* m, double* v, double M_star)
{
    double p[3];
    mass_weighted_velocity(N, m, v, p, NULL);
    for (int i = 0; i < N; ++i)
        for (int k = 0; k < 3; ++k) v[3 * i + k] += p[k] / M_star;
}

/* ---- O2: critical radius, Eq. 1 ---------------------------------------------
 *   r_crit,i = max(n1 R_H,i , n2 dt v_i),  R_H,i = a_i (m_i / 3 M_star)^(1/3).
 * Readings G2b/G2c: a_i from vis-viva with the stored v and mu = G M_star (a_i = r_i when that
 * is not a positive finite number); v_i = sqrt(G M_star / a_i).                               */
void oracle_rcrit(int N, const double* m, const double* x, const double* v,
                  const oracle_params* p, double* rcrit, double* semi, double* vkep)
{
    const double mu = p->G * p->M_star;
    for (int i = 0; i < N; ++i) {
        const double* xi = x + 3 * i;
        const double* vi = v + 3 * i;
        double r  = sqrt(xi[0] * xi[0] + xi[1] * xi[1] + xi[2] * xi[2]);
        double v2 = vi[0] * vi[0] + vi[1] * vi[1] + vi[2] * vi[2];
        double a  = 1.0 / (2.0 / r - v2 / mu);
        if (!(a > 0.0) || !isfinite(a)) a = r;
        double RH = a * cbrt(m[i] / (3.0 * p->M_star));
        double vk = sqrt(mu / a);
        double rc = fmax(p->n1 * RH, p->n2 * p->dt_rcrit * vk);
        if (rcrit) rcrit[i] = rc;
        if (semi)  semi[i]  = a;
        if (vkep)  vkep[i]  = vk;
    }
}

/* ---- O3: pair radius, reading G2 ----------------------------------------------------------- */
double oracle_pair_rcrit(const oracle_params* p, double mi, double mj,
                         double rci, double rcj, double ai, double aj,
                         double vki, double vkj)
{
    if (p->pair_rule == ORACLE_PAIR_MUTUAL_HILL) {
        double hill = p->n1 * cbrt((mi + mj) / (3.0 * p->M_star)) * (0.5 * (ai + aj));
        double vel  = p->n2 * p->dt_rcrit * fmax(vki, vkj);
        return fmax(hill, vel);
    }
    return fmax(rci, rcj);
}

/* ---- O2-O5: the kick acceleration (north_star; "the N^2 gravitational force
 * terms") ---------------------------------------------------------------------------------- */
/* TP2 mode ("the giant planets feel the forces of the planetesimals, but the
 * planetesimals do not feel each other"; reading R9): does the pair (i, j) interact at all? */
static int interacts(const oracle_params* p, int i, int j)
{
    return p->n_big < 0 || i < p->n_big || j < p->n_big;
}

/* O5 for one body i: sum over j != i, j ascending, Neumaier-compensated. */
static void accel_one(int N, const double* m, const double* x, const oracle_params* p,
                      const double* rc, const double* sa, const double* vk, int i, double out[3])
{
    nsum a[3] = {{0, 0}, {0, 0}, {0, 0}};
    for (int j = 0; j < N; ++j) {
        if (j == i || !interacts(p, i, j)) continue;
        double dx = x[3 * j + 0] - x[3 * i + 0];
        double dy = x[3 * j + 1] - x[3 * i + 1];
        double dz = x[3 * j + 2] - x[3 * i + 2];
        double r2 = dx * dx + dy * dy + dz * dz;
        double r  = sqrt(r2);
        if (!(r > 0.0)) continue;                     /* coincident bodies: W = 0 */
        double rcij = oracle_pair_rcrit(p, m[i], m[j], rc[i], rc[j], sa[i], sa[j], vk[i], vk[j]);
        double W = oracle_weight(r, rcij, p->weight_mode);
        if (W == 0.0) continue;
        double s = p->G * m[j] * W / (r2 * r);
        nsum_add(&a[0], s * dx);
        nsum_add(&a[1], s * dy);
        nsum_add(&a[2], s * dz);
    }
    for (int k = 0; k < 3; ++k) out[k] = nsum_value(&a[k]);
}

void oracle_accel(int N, const double* m, const double* x, const double* v,
                  const oracle_params* p, double* acc)
{
    double* rc = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* sa = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* vk = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    oracle_rcrit(N, m, x, v, p, rc, sa, vk);
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < N; ++i) accel_one(N, m, x, p, rc, sa, vk, i, acc + 3 * i);
    free(rc); free(sa); free(vk);
}

/* The same for the nsel bodies sel[0..nsel) only (sampled outputs at sizes where all N^2 pairs take too
 * long on a CPU): acc[k] = a_{sel[k]}.                                                                */
void oracle_accel_subset(int N, const double* m, const double* x, const double* v,
                         const oracle_params* p, int nsel, const int* sel, double* acc)
{
    double* rc = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* sa = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* vk = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    oracle_rcrit(N, m, x, v, p, rc, sa, vk);
#pragma omp parallel for schedule(dynamic, 4)
    for (int k = 0; k < nsel; ++k) accel_one(N, m, x, p, rc, sa, vk, sel[k], acc + 3 * k);
    free(rc); free(sa); free(vk);
}

/* O6 restricted to the pairs that touch one of the bodies sel[0..nsel): every (i, j), i = sel[k], j != i,
 * with r_ij < r_crit,ij, written as (min, max); a pair with both ends selected appears twice.         */
void oracle_encounter_pairs_subset(int N, const double* m, const double* x, const double* v,
                                   const oracle_params* p, int nsel, const int* sel,
                                   int* pairs, int cap, int* count)
{
    double* rc = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* sa = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* vk = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    oracle_rcrit(N, m, x, v, p, rc, sa, vk);
    int n = 0;
    for (int k = 0; k < nsel; ++k) {
        int i = sel[k];
        for (int j = 0; j < N; ++j) {
            if (j == i || !interacts(p, i, j)) continue;
            double dx = x[3 * j + 0] - x[3 * i + 0];
            double dy = x[3 * j + 1] - x[3 * i + 1];
            double dz = x[3 * j + 2] - x[3 * i + 2];
            double r  = sqrt(dx * dx + dy * dy + dz * dz);
            double rcij = oracle_pair_rcrit(p, m[i], m[j], rc[i], rc[j], sa[i], sa[j], vk[i], vk[j]);
            if (r < rcij) {
                if (n < cap && pairs) { pairs[2 * n] = i < j ? i : j; pairs[2 * n + 1] = i < j ? j : i; }
                ++n;
            }
        }
    }
    *count = n;
    free(rc); free(sa); free(vk);
}

/* ---- O6: encounter set, strict r < r_crit,ij (reading G6), PAPER.md:55 --------------------- */
void oracle_encounter_pairs(int N, const double* m, const double* x, const double* v,
                            const oracle_params* p, int* pairs, int cap, int* count)
{
    double* rc = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* sa = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* vk = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    oracle_rcrit(N, m, x, v, p, rc, sa, vk);
    int n = 0;
    for (int i = 0; i < N; ++i) {
        for (int j = i + 1; j < N; ++j) {
            if (!interacts(p, i, j)) continue;
            double dx = x[3 * j + 0] - x[3 * i + 0];
            double dy = x[3 * j + 1] - x[3 * i + 1];
            double dz = x[3 * j + 2] - x[3 * i + 2];
            double r  = sqrt(dx * dx + dy * dy + dz * dz);
            double rcij = oracle_pair_rcrit(p, m[i], m[j], rc[i], rc[j], sa[i], sa[j], vk[i], vk[j]);
            if (r < rcij) {
                if (n < cap && pairs) { pairs[2 * n] = i; pairs[2 * n + 1] = j; }
                ++n;
            }
        }
    }
    *count = n;
    free(rc); free(sa); free(vk);
}

/* ---- O7: velocity update -------------------------------------------------------------------- */
void oracle_kick(int N, const double* m, const double* x, double* v,
                 const oracle_params* p, double tau, double* acc_out)
{
    double* a = (double*)malloc(sizeof(double) * 3 * (size_t)(N > 0 ? N : 1));
    oracle_accel(N, m, x, v, p, a);
    for (int i = 0; i < 3 * N; ++i) v[i] += tau * a[i];
    if (acc_out) for (int i = 0; i < 3 * N; ++i) acc_out[i] = a[i];
    free(a);
}

/* ---- O8: Sun-kick of the democratic-heliocentric split (reading G3) ------------------------ */
void oracle_sunkick(int N, const double* m, double* x, const double* v,
                    const oracle_params* p, double tau)
{
    double s[3];
    mass_weighted_velocity(N, m, v, s, NULL);
    for (int i = 0; i < N; ++i)
        for (int k = 0; k < 3; ++k) x[3 * i + k] += tau * (s[k] / p->M_star);
}

/* ---- O9: Kepler drift, PAPER.md:43 ("Kepler orbit solver is always performed in double
 * precision"), reading G4: the exact two-body map about mu = G M_star.
 *
 * Anomaly-difference form.  With r0 = |x0|, u = x0.v0, alpha = 2 mu/r0 - |v0|^2 = mu/a:
 *  ellipse (alpha > 0): n = sqrt(mu/a^3); solve
 *        dE - (1 - r0/a) sin dE + (u/(n a^2)) (1 - cos dE) = n dt                      (K)
 *     f = 1 - (a/r0)(1 - cos dE),             g = dt - (dE - sin dE)/n,
 *     r = a + (r0 - a) cos dE + (u/(n a)) sin dE,
 *     fdot = -a^2 n sin dE /(r r0),           gdot = 1 - (a/r)(1 - cos dE).
 *  hyperbola (alpha < 0): b = -a > 0, nu = sqrt(mu/b^3); the same with
 *     sin -> sinh, (1 - cos) -> -(cosh - 1), i.e. with the functions
 *     G1 = sinh dH/sqrt(beta), G2 = (cosh dH - 1)/beta, G3 = (sinh dH - dH)/beta^(3/2), beta = -alpha:
 *        r0 G1 + u G2 + mu G3 = dt,   f = 1 - mu G2/r0,  g = dt - mu G3,
 *        r = r0 cosh dH + u G1 + mu G2,  fdot = -mu G1/(r r0),  gdot = 1 - mu G2/r.
 *  parabola (alpha = 0): G1 = s, G2 = s^2/2, G3 = s^3/6.
 * x = f x0 + g v0, v = fdot x0 + gdot v0.  The root is unique (the left side is strictly
 * increasing: its derivative is r/a resp. r/sqrt(beta) > 0); Newton with a bisection guard.     */

typedef double (*kep_fn)(double xx, const double* c, double* deriv);

static double kep_ell(double E, const double* c, double* d)
{   /* c = {EC, ES, M}: E - EC sin E + ES (1 - cos E) - M */
    double sE = sin(E), cE = cos(E);
    *d = 1.0 - c[0] * cE + c[1] * sE;
    return E - c[0] * sE + c[1] * (1.0 - cE) - c[2];
}
static double kep_hyp(double H, const double* c, double* d)
{   /* c = {r0, u, mu, sqrt(beta), beta, dt} */
    double sh = sinh(H), ch = cosh(H);
    double G1 = sh / c[3], G2 = (ch - 1.0) / c[4], G3 = (sh - H) / (c[4] * c[3]);
    *d = (c[0] * ch + c[1] * G1 + c[2] * G2) / c[3];
    return c[0] * G1 + c[1] * G2 + c[2] * G3 - c[5];
}
static double kep_par(double s, const double* c, double* d)
{   /* c = {r0, u, mu, dt} */
    *d = c[0] + c[1] * s + 0.5 * c[2] * s * s;
    return c[0] * s + 0.5 * c[1] * s * s + c[2] * s * s * s / 6.0 - c[3];
}

/* guarded Newton on a strictly increasing function, root bracketed in [lo, hi] */
static int solve_increasing(kep_fn F, const double* c, double lo, double hi, double x0, double* root)
{
    double xx = x0;
    if (!(xx > lo && xx < hi)) xx = 0.5 * (lo + hi);
    for (int it = 0; it < 200; ++it) {
        double d, f = F(xx, c, &d);
        if (f == 0.0) { *root = xx; return 0; }
        if (f > 0.0) hi = xx; else lo = xx;
        double xn = xx - f / d;
        if (!(xn > lo && xn < hi)) xn = 0.5 * (lo + hi);
        double step = fabs(xn - xx);
        xx = xn;
        if (step <= 1e-16 * fmax(1.0, fabs(xx)) || hi - lo <= 4e-16 * fmax(1.0, fabs(xx))) {
            *root = xx; return 0;
        }
    }
    *root = xx;
    return -1;
}

int oracle_kepler_drift_one(double mu, double dt, double x[3], double v[3])
{
    const double TWO_PI = 6.283185307179586476925286766559;
    double r0 = sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
    double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    double u  = x[0] * v[0] + x[1] * v[1] + x[2] * v[2];
    double alpha = 2.0 * mu / r0 - v2;
    double f, g, fd, gd;
    int rcode = 0;

    if (dt == 0.0) return 0;

    if (alpha > 0.0) {
        double a  = mu / alpha;
        double n  = sqrt(mu / (a * a * a));
        double EC = 1.0 - r0 / a;
        double ES = u / (n * a * a);
        double M  = n * dt;
        double k  = floor(M / TWO_PI + 0.5);          /* whole revolutions */
        double Mr = M - k * TWO_PI;
        double c[3] = {EC, ES, Mr};
        double dE;
        rcode = solve_increasing(kep_ell, c, Mr - 3.2, Mr + 3.2, Mr, &dE);
        double sE = sin(dE), cE = cos(dE);
        double h  = sin(0.5 * dE);
        double omc = 2.0 * h * h;                      /* 1 - cos dE */
        double r  = a + (r0 - a) * cE + (u / (n * a)) * sE;
        f  = 1.0 - (a / r0) * omc;
        g  = dt - ((dE - sE) + k * TWO_PI) / n;
        fd = -a * a * n * sE / (r * r0);
        gd = 1.0 - (a / r) * omc;
    } else if (alpha < 0.0) {
        double beta = -alpha, sb = sqrt(beta);
        double c[6] = {r0, u, mu, sb, beta, dt};
        /* F(0) = -dt: bracket the root by doubling away from 0 in the direction of dt */
        double lo = 0.0, hi = 0.0, d;
        int guard = 0;
        if (dt > 0.0) { hi = 0.5; while (kep_hyp(hi, c, &d) < 0.0 && ++guard < 64) { lo = hi; hi *= 2.0; } }
        else          { lo = -0.5; while (kep_hyp(lo, c, &d) > 0.0 && ++guard < 64) { hi = lo; lo *= 2.0; } }
        if (guard >= 64) return -1;
        double H;
        rcode = solve_increasing(kep_hyp, c, lo, hi, 0.5 * (lo + hi), &H);
        double sh = sinh(H), ch = cosh(H);
        double hh = sinh(0.5 * H);
        double chm1 = 2.0 * hh * hh;                   /* cosh H - 1 */
        double G1 = sh / sb, G2 = chm1 / beta, G3 = (sh - H) / (beta * sb);
        double r  = r0 * ch + u * G1 + mu * G2;
        f  = 1.0 - mu * G2 / r0;
        g  = dt - mu * G3;
        fd = -mu * G1 / (r * r0);
        gd = 1.0 - mu * G2 / r;
    } else {
        double c[4] = {r0, u, mu, dt};
        double lo = 0.0, hi = 0.0, d, s;
        int guard = 0;
        if (dt > 0.0) { hi = dt / r0; while (kep_par(hi, c, &d) < 0.0 && ++guard < 64) { lo = hi; hi *= 2.0; } }
        else          { lo = dt / r0; while (kep_par(lo, c, &d) > 0.0 && ++guard < 64) { hi = lo; lo *= 2.0; } }
        if (guard >= 64) return -1;
        rcode = solve_increasing(kep_par, c, lo, hi, dt / r0, &s);
        double G1 = s, G2 = 0.5 * s * s, G3 = s * s * s / 6.0;
        double r  = r0 + u * G1 + mu * G2;
        f  = 1.0 - mu * G2 / r0;
        g  = dt - mu * G3;
        fd = -mu * G1 / (r * r0);
        gd = 1.0 - mu * G2 / r;
    }

    double nx[3], nv[3];
    for (int k = 0; k < 3; ++k) {
        nx[k] = f * x[k] + g * v[k];
        nv[k] = fd * x[k] + gd * v[k];
    }
    for (int k = 0; k < 3; ++k) { x[k] = nx[k]; v[k] = nv[k]; }
    return rcode;
}

int oracle_drift(int N, double* x, double* v, const oracle_params* p, double dt)
{
    const double mu = p->G * p->M_star;
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
    for (int i = 0; i < N; ++i)
        if (oracle_kepler_drift_one(mu, dt, x + 3 * i, v + 3 * i) != 0) ++bad;
    return bad ? -1 : 0;
}

/* ---- O10: one level-0 step ("the symplectic integrator with a fixed step size
 * wherein bodies revolve around the central mass (level 0)"; splitting per reading G3) ------ */
static int sds(int N, const double* m, double* x, double* v, const oracle_params* p, double dt)
{
    oracle_sunkick(N, m, x, v, p, 0.5 * dt);
    int rc = oracle_drift(N, x, v, p, dt);
    oracle_sunkick(N, m, x, v, p, 0.5 * dt);
    return rc;
}

int oracle_step(int N, const double* m, double* x, double* v,
                const oracle_params* p, double dt)
{
    oracle_kick(N, m, x, v, p, 0.5 * dt, NULL);
    int rc = sds(N, m, x, v, p, dt);
    oracle_kick(N, m, x, v, p, 0.5 * dt, NULL);
    return rc;
}

int oracle_run(int N, const double* m, double* x, double* v,
               const oracle_params* p, double dt, int nsteps)
{
    int rc = 0;
    if (nsteps <= 0) return 0;
    oracle_kick(N, m, x, v, p, 0.5 * dt, NULL);
    for (int s = 0; s < nsteps; ++s) {
        if (sds(N, m, x, v, p, dt) != 0) rc = -1;
        oracle_kick(N, m, x, v, p, (s + 1 < nsteps) ? dt : 0.5 * dt, NULL);
    }
    return rc;
}

/* ---- NEXT-1: the encounter complement, reading R11 -------------------
 * "a changeover function smoothly switches" a pair between the fixed-step level-0 integrator and
 * the close-encounter integrator; encounter forces in double precision.  Hybrid symplectic split
 * (Chambers 1999; democratic heliocentric as G3):
 *   H_A = sum_i (|p_i|^2/2m_i - G M m_i/r_i) - sum_{i<j} G m_i m_j (1 - K(r_ij))/r_ij   Kepler + encounters
 *   H_B = - sum_{i<j} G m_i m_j K(r_ij)/r_ij                                            the level-0 kick
 *   H_C = |sum_i p_i|^2 / 2M                                                            the Sun-kick
 *   step = B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2).
 * B is oracle_kick with weight_mode = 1 (W = K - r K', the gradient of H_B).  A has no closed form once a pair
 * is inside its zone; the oracle integrates the flow of H_A for ALL bodies numerically (classical RK4, nsub
 * equal substeps: plain and slow, no encounter groups, no pair lists), with the pair weight
 * Wc = 1 - W = (1 - K) + r K' and r_crit,ij held at the values of the opening force evaluation.  With no pair
 * inside a zone Wc = 0 everywhere and A is the Kepler drift, so the step reduces to oracle_step.           */
static void rhs_A_s(int N, const double* m, const oracle_params* p, const double* rc, const double* sa,
                    const double* vk, const double* x, const double* v, double* dx, double* dv, double rscale);
static void rhs_A(int N, const double* m, const oracle_params* p, const double* rc, const double* sa,
                  const double* vk, const double* x, const double* v, double* dx, double* dv)
{
    rhs_A_s(N, m, p, rc, sa, vk, x, v, dx, dv, 1.0);
}
/* rscale: the critical radii are multiplied by it (1 for the two-level step; 1 / F^(L-1) for the innermost level of the
 * multi-level step, reading R16) */
static void rhs_A_s(int N, const double* m, const oracle_params* p, const double* rc, const double* sa,
                    const double* vk, const double* x, const double* v, double* dx, double* dv, double rscale)
{
    const double mu = p->G * p->M_star;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        const double* xi = x + 3 * i;
        double r2 = xi[0] * xi[0] + xi[1] * xi[1] + xi[2] * xi[2];
        double r  = sqrt(r2);
        double a[3] = {-mu * xi[0] / (r2 * r), -mu * xi[1] / (r2 * r), -mu * xi[2] / (r2 * r)};
        for (int j = 0; j < N; ++j) {
            if (j == i || !interacts(p, i, j)) continue;
            double d[3] = {x[3 * j] - xi[0], x[3 * j + 1] - xi[1], x[3 * j + 2] - xi[2]};
            double q2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            double q  = sqrt(q2);
            if (!(q > 0.0)) continue;
            double rcij = rscale * oracle_pair_rcrit(p, m[i], m[j], rc[i], rc[j], sa[i], sa[j], vk[i], vk[j]);
            double Wc = 1.0 - oracle_weight(q, rcij, 1);
            if (Wc == 0.0) continue;
            double s = p->G * m[j] * Wc / (q2 * q);
            a[0] += s * d[0]; a[1] += s * d[1]; a[2] += s * d[2];
        }
        for (int k = 0; k < 3; ++k) { dx[3 * i + k] = v[3 * i + k]; dv[3 * i + k] = a[k]; }
    }
}

/* A(dt): nsub RK4 substeps of the flow of H_A with the given (fixed) critical radii. */
void oracle_encounter_drift(int N, const double* m, double* x, double* v, const oracle_params* p,
                            const double* rc, const double* sa, const double* vk, double dt, int nsub)
{
    size_t n3 = 3 * (size_t)(N > 0 ? N : 1);
    double* buf = (double*)malloc(sizeof(double) * n3 * 10);
    double *k1x = buf, *k1v = buf + n3, *k2x = buf + 2 * n3, *k2v = buf + 3 * n3, *k3x = buf + 4 * n3,
           *k3v = buf + 5 * n3, *k4x = buf + 6 * n3, *k4v = buf + 7 * n3, *tx = buf + 8 * n3, *tv = buf + 9 * n3;
    double h = dt / nsub;
    for (int s = 0; s < nsub; ++s) {
        rhs_A(N, m, p, rc, sa, vk, x, v, k1x, k1v);
        for (int q = 0; q < 3 * N; ++q) { tx[q] = x[q] + 0.5 * h * k1x[q]; tv[q] = v[q] + 0.5 * h * k1v[q]; }
        rhs_A(N, m, p, rc, sa, vk, tx, tv, k2x, k2v);
        for (int q = 0; q < 3 * N; ++q) { tx[q] = x[q] + 0.5 * h * k2x[q]; tv[q] = v[q] + 0.5 * h * k2v[q]; }
        rhs_A(N, m, p, rc, sa, vk, tx, tv, k3x, k3v);
        for (int q = 0; q < 3 * N; ++q) { tx[q] = x[q] + h * k3x[q]; tv[q] = v[q] + h * k3v[q]; }
        rhs_A(N, m, p, rc, sa, vk, tx, tv, k4x, k4v);
        for (int q = 0; q < 3 * N; ++q) {
            x[q] += h / 6.0 * (k1x[q] + 2.0 * k2x[q] + 2.0 * k3x[q] + k4x[q]);
            v[q] += h / 6.0 * (k1v[q] + 2.0 * k2v[q] + 2.0 * k3v[q] + k4v[q]);
        }
    }
    free(buf);
}

/* A(dt) with an error-controlled integrator: Gragg-Bulirsch-Stoer extrapolation ("the Bulirsch-Stoer
 * integrator (level 1)"; Stoer & Bulirsch 1980, sect. 7.2.14; the scheme itself is textbook material and is restated
 * here, reading R15).  One macro step of size H from y = (x, v):
 *   modified midpoint with n_k = 2 (k + 1) substeps h = H / n_k, k = 0 .. 7:
 *     z_0 = y, z_1 = z_0 + h f(z_0), z_{m+1} = z_{m-1} + 2 h f(z_m), S_k = (z_n + z_{n-1} + h f(z_n)) / 2,
 *   polynomial extrapolation in h^2 (Aitken-Neville):
 *     T_{k,0} = S_k,  T_{k,j} = T_{k,j-1} + (T_{k,j-1} - T_{k-1,j-1}) / ((n_k / n_{k-j})^2 - 1),
 *   error of row k: max over bodies of max(|dx_i| / |x_i|, |dv_i| / |v_i|) with d = T_{k,k} - T_{k,k-1} (vector norms);
 *   accepted as soon as it is <= tol (k >= 1); if row 7 fails, H is halved and the step repeated.  After a step that
 *   took row k the next H is 2 H (k <= 3), H (k <= 5) or H / 2, cut to what is left of dt.
 * All N bodies form ONE system (no groups, no lists): the oracle of the A-flow is its converged solution.
 * stats (may be NULL): [0] macro steps accepted, [1] rejected, [2] right-hand sides.  Returns 0, or -1 if H fell
 * below |dt| 2^-40 without convergence (the state is then the last accepted one).                                 */
static int drift_bs(int N, const double* m, double* x, double* v, const oracle_params* p, const double* rc,
                    const double* sa, const double* vk, double dt, double tol, long long* stats, double rscale);
int oracle_encounter_drift_bs(int N, const double* m, double* x, double* v, const oracle_params* p,
                              const double* rc, const double* sa, const double* vk, double dt, double tol, long long* stats)
{
    return drift_bs(N, m, x, v, p, rc, sa, vk, dt, tol, stats, 1.0);
}
static int drift_bs(int N, const double* m, double* x, double* v, const oracle_params* p, const double* rc,
                    const double* sa, const double* vk, double dt, double tol, long long* stats, double rscale)
{
    enum { KMAX = 8 };
    size_t n3 = 3 * (size_t)(N > 0 ? N : 1);
    double* buf = (double*)malloc(sizeof(double) * n3 * (8 + 4 * KMAX));
    double *f0x = buf, *f0v = buf + n3, *z0x = buf + 2 * n3, *z0v = buf + 3 * n3, *z1x = buf + 4 * n3, *z1v = buf + 5 * n3,
           *fx = buf + 6 * n3, *fv = buf + 7 * n3;
    double* Tx[2][KMAX]; double* Tv[2][KMAX];                     /* two rows of the tableau */
    for (int r = 0; r < 2; ++r)
        for (int j = 0; j < KMAX; ++j) { Tx[r][j] = buf + (8 + (2 * r) * KMAX + j) * n3; Tv[r][j] = buf + (8 + (2 * r + 1) * KMAX + j) * n3; }
    long long acc = 0, rej = 0, nf = 0;
    int rcode = 0;
    double t = 0.0, H = dt;
    const double T = fabs(dt);
    while (fabs(t) < T * (1.0 - 1.0e-14) && T > 0.0) {
        if (fabs(t + H) > T) H = dt - t;
        rhs_A_s(N, m, p, rc, sa, vk, x, v, f0x, f0v, rscale); ++nf;
        int done = -1;
        for (int k = 0; k < KMAX && done < 0; ++k) {
            const int nk = 2 * (k + 1);
            const double h = H / nk;
            const int cur = k & 1, prev = cur ^ 1;
            for (size_t q = 0; q < 3 * (size_t)N; ++q) { z0x[q] = x[q]; z0v[q] = v[q]; z1x[q] = x[q] + h * f0x[q]; z1v[q] = v[q] + h * f0v[q]; }
            for (int s = 1; s < nk; ++s) {
                rhs_A_s(N, m, p, rc, sa, vk, z1x, z1v, fx, fv, rscale); ++nf;
                for (size_t q = 0; q < 3 * (size_t)N; ++q) {
                    double nx = z0x[q] + 2.0 * h * fx[q], nv = z0v[q] + 2.0 * h * fv[q];
                    z0x[q] = z1x[q]; z0v[q] = z1v[q]; z1x[q] = nx; z1v[q] = nv;
                }
            }
            rhs_A_s(N, m, p, rc, sa, vk, z1x, z1v, fx, fv, rscale); ++nf;
            for (size_t q = 0; q < 3 * (size_t)N; ++q) {
                Tx[cur][0][q] = 0.5 * (z1x[q] + z0x[q] + h * fx[q]);
                Tv[cur][0][q] = 0.5 * (z1v[q] + z0v[q] + h * fv[q]);
            }
            for (int j = 1; j <= k; ++j) {
                const double ratio = (double)nk / (double)(2 * (k - j + 1));
                const double den = ratio * ratio - 1.0;
                for (size_t q = 0; q < 3 * (size_t)N; ++q) {
                    Tx[cur][j][q] = Tx[cur][j - 1][q] + (Tx[cur][j - 1][q] - Tx[prev][j - 1][q]) / den;
                    Tv[cur][j][q] = Tv[cur][j - 1][q] + (Tv[cur][j - 1][q] - Tv[prev][j - 1][q]) / den;
                }
            }
            if (k >= 1) {
                double err = 0.0;
                for (int i = 0; i < N; ++i) {
                    double dx2 = 0, dv2 = 0, x2 = 0, v2 = 0;
                    for (int c = 0; c < 3; ++c) {
                        double a = Tx[cur][k][3 * i + c], b = Tv[cur][k][3 * i + c];
                        double da = a - Tx[cur][k - 1][3 * i + c], db = b - Tv[cur][k - 1][3 * i + c];
                        dx2 += da * da; dv2 += db * db; x2 += a * a; v2 += b * b;
                    }
                    double ex = sqrt(dx2 / x2), ev = sqrt(dv2 / v2);
                    if (!(ex <= err)) err = ex;               /* NaN counts as "not converged" */
                    if (!(ev <= err)) err = ev;
                }
                if (err <= tol) done = k;
            }
        }
        if (done < 0) {
            ++rej;
            H *= 0.5;
            if (fabs(H) < T * 9.094947017729282e-13) { rcode = -1; break; }
            continue;
        }
        for (size_t q = 0; q < 3 * (size_t)N; ++q) { x[q] = Tx[done & 1][done][q]; v[q] = Tv[done & 1][done][q]; }
        t += H; ++acc;
        H = (done <= 3) ? 2.0 * H : ((done <= 5) ? H : 0.5 * H);
    }
    if (stats) { stats[0] += acc; stats[1] += rej; stats[2] += nf; }
    free(buf);
    return rcode;
}

/* The hybrid step of reading R11 with A(dt) integrated to the tolerance tol by oracle_encounter_drift_bs. */
int oracle_step_hybrid_bs(int N, const double* m, double* x, double* v, const oracle_params* p, double dt, double tol,
                          long long* stats)
{
    if (p->weight_mode != 1 || !(tol > 0.0)) return -1;
    double* rc = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* sa = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* vk = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    oracle_rcrit(N, m, x, v, p, rc, sa, vk);              /* the radii of the opening force evaluation */
    oracle_kick(N, m, x, v, p, 0.5 * dt, NULL);
    oracle_sunkick(N, m, x, v, p, 0.5 * dt);
    if (stats) { stats[0] = 0; stats[1] = 0; stats[2] = 0; }
    int r = oracle_encounter_drift_bs(N, m, x, v, p, rc, sa, vk, dt, tol, stats);
    oracle_sunkick(N, m, x, v, p, 0.5 * dt);
    oracle_kick(N, m, x, v, p, 0.5 * dt, NULL);
    free(rc); free(sa); free(vk);
    return r;
}

/* ---- NEXT-3, second half: multi-level changeover, reading R16 ---------------------------
 * "a hierarchical method that uses multiple changeover functions ... instead of switching directly to
 * the Bulirsch-Stoer method, another symplectic integration step with a reduced time step can be applied in between";
 * "the number of levels and the number of sub-steps".  Grimm et al. 2022 is not in the container; the
 * reading (recursive shells as in Duncan et al. 1998, whom the paper cites, with Chambers' K on every level):
 *   L levels of changeover, S sub-steps per level, radius ratio F:  level l uses r_crit,ij / F^l and the step dt / S^l.
 *   W_l(r) = weight(r, r_crit,ij / F^l) (K - r K', reading R10), W_{-1} = 0.  The pair potential V = -G m_i m_j / r is
 *   cut into shells  V = W_0 V + sum_{l=1}^{L-1} (W_l - W_{l-1}) V + (1 - W_{L-1}) V  (as forces; the weights add to 1):
 *   shell 0 is the level-0 kick (step dt), shell l a kick with the step dt / S^l, the remainder stays with the Kepler
 *   terms in the Bulirsch-Stoer integration (level L) over dt / S^(L-1).  Recursively, flow_l(tau) of
 *   H_Kep + (1 - W_{l-1}) V:   flow_L(tau) = Bulirsch-Stoer;   flow_l(tau) = [ kick_l(h/2) flow_{l+1}(h) kick_l(h/2) ]^S,
 *   h = tau / S;   step = B(dt/2) C(dt/2) flow_1(dt) C(dt/2) B(dt/2).
 * L = 1 is the two-level hybrid step of R11 / R15.  Critical radii: those of the opening force evaluation.         */
double oracle_level_weight(double r, double rcrit, int l, int L, double F)
{
    double lo = 0.0, hi = 1.0, sc = 1.0;
    for (int k = 0; k < l - 1; ++k) sc /= F;
    if (l >= 1) lo = oracle_weight(r, rcrit * sc, 1);            /* W_{l-1} */
    if (l < L)  hi = oracle_weight(r, rcrit * (l >= 1 ? sc / F : 1.0), 1);   /* W_l; l == L: the remainder 1 - W_{L-1} */
    return hi - lo;
}

/* v_i += tau * sum_j G m_j w_l(r_ij) (x_j - x_i) / r_ij^3 with the shell weight of level l (1 <= l < L) */
static void shell_kick(int N, const double* m, const double* x, double* v, const oracle_params* p, const double* rc,
                       const double* sa, const double* vk, int l, int L, double F, double tau)
{
    double* a = (double*)calloc(3 * (size_t)(N > 0 ? N : 1), sizeof(double));
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        nsum s3[3] = {{0, 0}, {0, 0}, {0, 0}};
        for (int j = 0; j < N; ++j) {
            if (j == i || !interacts(p, i, j)) continue;
            double d[3] = {x[3 * j] - x[3 * i], x[3 * j + 1] - x[3 * i + 1], x[3 * j + 2] - x[3 * i + 2]};
            double q2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            double q  = sqrt(q2);
            if (!(q > 0.0)) continue;
            double rcij = oracle_pair_rcrit(p, m[i], m[j], rc[i], rc[j], sa[i], sa[j], vk[i], vk[j]);
            double wl = oracle_level_weight(q, rcij, l, L, F);
            if (wl == 0.0) continue;
            double s = p->G * m[j] * wl / (q2 * q);
            for (int k = 0; k < 3; ++k) nsum_add(&s3[k], s * d[k]);
        }
        for (int k = 0; k < 3; ++k) a[3 * i + k] = nsum_value(&s3[k]);
    }
    for (size_t q = 0; q < 3 * (size_t)N; ++q) v[q] += tau * a[q];
    free(a);
}

static int level_flow(int N, const double* m, double* x, double* v, const oracle_params* p, const double* rc,
                      const double* sa, const double* vk, int l, int L, int S, double F, double tau, double tol, long long* stats)
{
    if (l >= L) {
        double sc = 1.0;
        for (int k = 0; k < L - 1; ++k) sc /= F;
        return drift_bs(N, m, x, v, p, rc, sa, vk, tau, tol, stats, sc);
    }
    int rcode = 0;
    const double h = tau / S;
    for (int s = 0; s < S; ++s) {
        shell_kick(N, m, x, v, p, rc, sa, vk, l, L, F, 0.5 * h);
        if (level_flow(N, m, x, v, p, rc, sa, vk, l + 1, L, S, F, h, tol, stats) != 0) rcode = -1;
        shell_kick(N, m, x, v, p, rc, sa, vk, l, L, F, 0.5 * h);
    }
    return rcode;
}

int oracle_step_multilevel(int N, const double* m, double* x, double* v, const oracle_params* p, double dt,
                           int L, int S, double F, double tol, long long* stats)
{
    if (p->weight_mode != 1 || !(tol > 0.0) || L < 1 || S < 1 || !(F > 1.0)) return -1;
    double* rc = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* sa = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* vk = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    oracle_rcrit(N, m, x, v, p, rc, sa, vk);              /* the radii of the opening force evaluation */
    oracle_kick(N, m, x, v, p, 0.5 * dt, NULL);
    oracle_sunkick(N, m, x, v, p, 0.5 * dt);
    if (stats) { stats[0] = 0; stats[1] = 0; stats[2] = 0; }
    int r = level_flow(N, m, x, v, p, rc, sa, vk, 1, L, S, F, dt, tol, stats);
    oracle_sunkick(N, m, x, v, p, 0.5 * dt);
    oracle_kick(N, m, x, v, p, 0.5 * dt, NULL);
    free(rc); free(sa); free(vk);
    return r;
}

/* One hybrid step B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2); p->weight_mode must be 1.  Returns -1 otherwise. */
int oracle_step_hybrid(int N, const double* m, double* x, double* v, const oracle_params* p, double dt, int nsub)
{
    if (p->weight_mode != 1 || nsub < 1) return -1;
    double* rc = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* sa = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double* vk = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    oracle_rcrit(N, m, x, v, p, rc, sa, vk);              /* the radii of the opening force evaluation */
    oracle_kick(N, m, x, v, p, 0.5 * dt, NULL);
    oracle_sunkick(N, m, x, v, p, 0.5 * dt);
    oracle_encounter_drift(N, m, x, v, p, rc, sa, vk, dt, nsub);
    oracle_sunkick(N, m, x, v, p, 0.5 * dt);
    oracle_kick(N, m, x, v, p, 0.5 * dt, NULL);
    free(rc); free(sa); free(vk);
    return 0;
}

/* ---- O11: diagnostics, PAPER.md:111 (Delta E/E = E(t)/E(0) - 1, likewise L), reading G5 ---- */
void oracle_energy_angmom(int N, const double* m, const double* x, const double* v,
                          const oracle_params* p, double* E, double L[3])
{
    nsum kin = {0, 0}, sol = {0, 0}, pot = {0, 0};
    nsum P[3] = {{0, 0}, {0, 0}, {0, 0}}, Ls[3] = {{0, 0}, {0, 0}, {0, 0}};
    for (int i = 0; i < N; ++i) {
        const double* xi = x + 3 * i;
        const double* vi = v + 3 * i;
        double r  = sqrt(xi[0] * xi[0] + xi[1] * xi[1] + xi[2] * xi[2]);
        double v2 = vi[0] * vi[0] + vi[1] * vi[1] + vi[2] * vi[2];
        nsum_add(&kin, 0.5 * m[i] * v2);
        nsum_add(&sol, p->G * p->M_star * m[i] / r);
        for (int k = 0; k < 3; ++k) nsum_add(&P[k], m[i] * vi[k]);
        nsum_add(&Ls[0], m[i] * (xi[1] * vi[2] - xi[2] * vi[1]));
        nsum_add(&Ls[1], m[i] * (xi[2] * vi[0] - xi[0] * vi[2]));
        nsum_add(&Ls[2], m[i] * (xi[0] * vi[1] - xi[1] * vi[0]));
    }
    /* pair potential: per-i partial sums in parallel, then added in i order */
    double* part = (double*)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < N; ++i) {
        nsum q = {0, 0};
        for (int j = i + 1; j < N; ++j) {
            if (!interacts(p, i, j)) continue;
            double dx = x[3 * j + 0] - x[3 * i + 0];
            double dy = x[3 * j + 1] - x[3 * i + 1];
            double dz = x[3 * j + 2] - x[3 * i + 2];
            double r  = sqrt(dx * dx + dy * dy + dz * dz);
            nsum_add(&q, p->G * m[i] * m[j] / r);
        }
        part[i] = nsum_value(&q);
    }
    for (int i = 0; i < N; ++i) nsum_add(&pot, part[i]);
    free(part);

    double px = nsum_value(&P[0]), py = nsum_value(&P[1]), pz = nsum_value(&P[2]);
    nsum e = {0, 0};
    nsum_add(&e, nsum_value(&kin));
    nsum_add(&e, (px * px + py * py + pz * pz) / (2.0 * p->M_star));
    nsum_add(&e, -nsum_value(&sol));
    nsum_add(&e, -nsum_value(&pot));
    *E = nsum_value(&e);
    for (int k = 0; k < 3; ++k) L[k] = nsum_value(&Ls[k]);
}

/* ---- NEXT-4: perfect mergers at a step end (reading R13) ------------------------
 * Plain definition: brute force over all pairs for the collision graph, components by repeated
 * relabelling to the smallest index until nothing changes, member sums in ascending index.        */
int oracle_merge(int N, double* m, double* x, double* v, double* R, int* newidx)
{
    return oracle_merge_tp2(N, m, x, v, R, newidx, -1, (int*)0);
}

/* The same with TP2 mode's rule for which pairs exist (readings R9, R13): only pairs with i < n_big or
 * j < n_big can collide (small bodies do not see each other); n_big < 0: every pair.  *n_big_new (may be NULL): the big
 * bodies left, i.e. the survivors among the first n_big (two big bodies that merge leave one).                        */
int oracle_merge_tp2(int N, double* m, double* x, double* v, double* R, int* newidx, int n_big, int* n_big_new)
{
    if (n_big_new) *n_big_new = n_big;
    if (N <= 0) return 0;
    int* lab = (int*)malloc(sizeof(int) * (size_t)N);
    for (int i = 0; i < N; ++i) lab[i] = i;
    int changed = 1;
    while (changed) {
        changed = 0;
        for (int i = 0; i < N; ++i)
            for (int j = i + 1; j < N; ++j) {
                if (lab[i] == lab[j]) continue;
                if (n_big >= 0 && i >= n_big && j >= n_big) continue;
                double dx = x[3 * j + 0] - x[3 * i + 0];
                double dy = x[3 * j + 1] - x[3 * i + 1];
                double dz = x[3 * j + 2] - x[3 * i + 2];
                double r  = sqrt(dx * dx + dy * dy + dz * dz);
                if (r < R[i] + R[j]) {
                    int lo = lab[i] < lab[j] ? lab[i] : lab[j];
                    lab[i] = lo; lab[j] = lo;
                    changed = 1;
                }
            }
    }
    /* merge every component into its smallest index (lab[k] == k there) */
    for (int r = 0; r < N; ++r) {
        if (lab[r] != r) continue;
        int members = 0;
        nsum M = {0, 0}, V3 = {0, 0}, X[3] = {{0, 0}, {0, 0}, {0, 0}}, P[3] = {{0, 0}, {0, 0}, {0, 0}};
        for (int k = r; k < N; ++k) {
            if (lab[k] != r) continue;
            ++members;
            nsum_add(&M, m[k]);
            nsum_add(&V3, R[k] * R[k] * R[k]);
            for (int d = 0; d < 3; ++d) { nsum_add(&X[d], m[k] * x[3 * k + d]); nsum_add(&P[d], m[k] * v[3 * k + d]); }
        }
        if (members < 2) continue;
        double mt = nsum_value(&M);
        if (mt > 0.0)
            for (int d = 0; d < 3; ++d) { x[3 * r + d] = nsum_value(&X[d]) / mt; v[3 * r + d] = nsum_value(&P[d]) / mt; }
        m[r] = mt;
        R[r] = cbrt(nsum_value(&V3));
    }
    /* close up the arrays in order */
    int n = 0;
    int* where = (int*)malloc(sizeof(int) * (size_t)N);
    for (int i = 0; i < N; ++i) {
        if (lab[i] != i) continue;
        where[i] = n;
        m[n] = m[i]; R[n] = R[i];
        for (int d = 0; d < 3; ++d) { x[3 * n + d] = x[3 * i + d]; v[3 * n + d] = v[3 * i + d]; }
        ++n;
    }
    if (newidx) for (int i = 0; i < N; ++i) newidx[i] = where[lab[i]];
    if (n_big_new && n_big >= 0) {
        int nb = 0;
        for (int i = 0; i < N && i < n_big; ++i) nb += (lab[i] == i);
        *n_big_new = nb;
    }
    free(where);
    free(lab);
    return n;
}

/* ---- NEXT-4, refinement: collisions INSIDE the encounter integration (reading R14; oracle only so far) ----
 * The hybrid step of reading R11 with the collision pass of reading R13 applied after EVERY RK4 substep of the
 * A-flow instead of once per step: an overlap is acted on at the first substep end that shows it.  The merged body
 * inherits the frozen per-body quantities of the opening evaluation (r_crit,i, a_i, v_K,i) from the component's
 * smallest index; masses are the merged ones.  newidx (may be NULL) maps the bodies before the step to the bodies
 * after it.  R = 0 for every body reproduces oracle_step_hybrid bit for bit.  Returns N', or -1 on bad params.   */
int oracle_step_hybrid_collide(int N, double* m, double* x, double* v, double* R, const oracle_params* p,
                               double dt, int nsub, int* newidx)
{
    if (p->weight_mode != 1 || nsub < 1) return -1;
    size_t n1 = (size_t)(N > 0 ? N : 1);
    double* rc = (double*)malloc(sizeof(double) * n1);
    double* sa = (double*)malloc(sizeof(double) * n1);
    double* vk = (double*)malloc(sizeof(double) * n1);
    int* step_idx = (int*)malloc(sizeof(int) * n1);
    int* total = (int*)malloc(sizeof(int) * n1);
    for (int i = 0; i < N; ++i) total[i] = i;
    int n = N;
    oracle_rcrit(n, m, x, v, p, rc, sa, vk);
    oracle_kick(n, m, x, v, p, 0.5 * dt, NULL);
    oracle_sunkick(n, m, x, v, p, 0.5 * dt);
    for (int s = 0; s < nsub; ++s) {
        oracle_encounter_drift(n, m, x, v, p, rc, sa, vk, dt / nsub, 1);      /* one RK4 substep of the A-flow */
        int n_new = oracle_merge(n, m, x, v, R, step_idx);
        if (n_new < n) {
            int k = 0;                                   /* survivors appear in order of their smallest member */
            for (int i = 0; i < n; ++i)
                if (step_idx[i] == k) { rc[k] = rc[i]; sa[k] = sa[i]; vk[k] = vk[i]; ++k; }
            for (int i = 0; i < N; ++i) total[i] = step_idx[total[i]];
            n = n_new;
        }
    }
    oracle_sunkick(n, m, x, v, p, 0.5 * dt);
    oracle_kick(n, m, x, v, p, 0.5 * dt, NULL);
    if (newidx) for (int i = 0; i < N; ++i) newidx[i] = total[i];
    free(rc); free(sa); free(vk); free(step_idx); free(total);
    return n;
}
