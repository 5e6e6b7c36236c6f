/*
 * genga_oracle.h -- CPU FP64 oracle for the GENGA level-0 hot path.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this library.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_2309_08217_b200/ and neither imports the other.
 *
 * What it computes follows /root/reference/PAPER.md (arXiv 2309.08217) where
 * the paper speaks, and the readings G1..G11 of SURVEY.md section 8(c) /
 * DESIGN.md section 3 where it is silent.  Every function is the plain
 * definition written out: sqrt and divide, no rsqrt tricks, no blocking, no
 * reordering, j ascending, Neumaier-compensated sums.
 *
 * Layout: m[N]; x, v, a are [N][3] row-major doubles; all pointers are HOST
 * pointers.  x is heliocentric; v is the stored ("democratic", i.e.
 * barycentric) velocity unless a function says otherwise.
 *
 * Pin status (see tests/test_oracle_*.py, marked "not gpu"):
 *   oracle_changeover      pinned: limits, hand values, symmetry (G1 reading: "parity unpinned
 *                          by PAPER.md" for the CHOICE of K -- the paper prints no formula)
 *   oracle_rcrit           pinned: Eq. 1 by hand
 *   oracle_accel           pinned: hand 3-/4-body values, n-gon closed form, sum m a = 0,
 *                          torque = 0, 50-digit brute force
 *   oracle_encounter_pairs pinned: brute force, constructed r_crit(1 -+ 1e-9) cases
 *   oracle_drift           pinned: circular orbit, period return, scipy DOP853, invariants
 *   oracle_step/run        pinned: 2nd-order convergence to a DOP853 inertial-frame solution
 *   oracle_energy_angmom   pinned: two-body closed form, inertial-frame formula
 *   oracle_weight mode 1   pinned: hand value at y = 1/2, limits, -r^2 d/dr[K/r] by central
 *                          differences of the pinned K, two-body force = -grad of the potential
 *   oracle_step_hybrid     pinned: reduces to oracle_step without encounters, energy through a close
 *                          encounter (full E) vs the level-0-only step, dt^2 convergence to DOP853
 *   oracle_step_hybrid_bs  pinned: Kepler motion of one body against the closed-form drift, DOP853 on the A-flow of a deep
 *                          encounter, agreement with the converged RK4 substeps of oracle_step_hybrid, error falling
 *                          with tol, time reversal (reading R15: WHICH extrapolation scheme and step control GENGA's
 *                          Bulirsch-Stoer level uses is not printed; the A-flow itself is unique)
 *   oracle_step_multilevel pinned: the shell weights add to 1 and are each >= 0, hand value of a shell; L = 1 is
 *                          oracle_step_hybrid_bs bit for bit; without encounters it is oracle_step; S = 1 with any L is
 *                          the two-level step to the integration tolerance; second-order convergence to the DOP853
 *                          N-body solution through an encounter; energy through the encounter against the level count
 *                          (reading R16: the level structure of Grimm et al. 2022 is NOT in PAPER.md -- parity unpinned
 *                          by the paper for that choice)
 *   TP2 mode (n_big >= 0)  pinned: hand 3-body values, full-minus-subset identity against the
 *                          pinned all-pairs path, sum m a = 0, bounded dt^2 energy error
 *   oracle_merge(_tp2)     pinned: inelastic-collision identities (dT = mu u^2/2, dL = mu x_rel x v_rel),
 *                          hand values (pair, chain, strictness, massless), scipy connected components,
 *                          conserved extensive sums (reading R13: WHEN collisions are looked for is a
 *                          reading -- the paper does not say; "parity unpinned by PAPER.md" for that choice)
 *   oracle_step_hybrid_collide  pinned: R = 0 is oracle_step_hybrid bit for bit, free-body closed forms,
 *                          impact parameter, pass-through vs step-end pass (reading R14; no GPU counterpart yet)
 */
#ifndef GENGA_ORACLE_H
#define GENGA_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

enum { ORACLE_PAIR_MAX = 0, ORACLE_PAIR_MUTUAL_HILL = 1 };

typedef struct {
    double G;         /* gravitational constant in the caller's units                */
    double M_star;    /* central mass                                                */
    double n1, n2;    /* Eq. 1 constants (3 and 0.4)                    */
    double dt_rcrit;  /* the dt of Eq. 1's second term (reading G8: the step dt)     */
    int    pair_rule; /* reading G2: how r_crit,ij follows from per-body quantities  */
    int    n_big;     /* TP2 mode (reading R9): a pair (i, j)
                         interacts iff i < n_big or j < n_big; n_big < 0: every pair
                         interacts.  Other pairs exert no force, are no encounter
                         candidates and carry no pair potential in E.              */
    int    weight_mode; /* 0: pair weight W = K (default); 1: W = K - r dK/dr, the gradient of
                           the K-weighted pair potential (reading R10, NEXT-3)  */
} oracle_params;

/* O4, reading G1 (PAPER.md:45 names Chambers 1999; formula not printed). */
double oracle_changeover(double r, double rcrit);
/* Pair weight W(r, r_crit): mode 0 = K, mode 1 = K - r dK/dr (reading R10).    */
double oracle_weight(double r, double rcrit, int mode);

/* O1: heliocentric velocities <-> stored barycentric ("democratic") ones.    */
void oracle_to_democratic(int N, const double* m, double* v, double M_star);
void oracle_to_heliocentric(int N, const double* m, double* v, double M_star);

/* O2, Eq. 1.  Outputs may be NULL.  semi = a_i, vkep = v_K,i. */
void oracle_rcrit(int N, const double* m, const double* x, const double* v,
                  const oracle_params* p, double* rcrit, double* semi, double* vkep);

/* O3: r_crit,ij from the per-body arrays returned by oracle_rcrit.           */
double oracle_pair_rcrit(const oracle_params* p, double mi, double mj,
                         double rci, double rcj, double ai, double aj,
                         double vki, double vkj);

/* O2-O5: a_i = sum_{j != i} G m_j K(r_ij, r_crit,ij) (x_j - x_i) / r_ij^3.   */
void oracle_accel(int N, const double* m, const double* x, const double* v,
                  const oracle_params* p, double* acc);

/* O5 / O6 for a sample of bodies sel[0..nsel): accelerations of those bodies; encounter pairs that
 * touch one of them, as (min, max), a pair with both ends in the sample listed twice.            */
void oracle_accel_subset(int N, const double* m, const double* x, const double* v,
                         const oracle_params* p, int nsel, const int* sel, double* acc);
void oracle_encounter_pairs_subset(int N, const double* m, const double* x, const double* v,
                                   const oracle_params* p, int nsel, const int* sel,
                                   int* pairs, int cap, int* count);

/* O6: { (i,j): i<j, r_ij < r_crit,ij } in lexicographic order.  Writes at most
 * cap pairs into pairs[cap][2]; *count receives the true total.              */
void oracle_encounter_pairs(int N, const double* m, const double* x, const double* v,
                            const oracle_params* p, int* pairs, int cap, int* count);

/* O7: v_i += tau * a_i (a from oracle_accel on the current state).  acc_out
 * may be NULL, else receives a.                                              */
void oracle_kick(int N, const double* m, const double* x, double* v,
                 const oracle_params* p, double tau, double* acc_out);

/* O8, reading G3: x_i += tau * (sum_j m_j v_j) / M_star.                     */
void oracle_sunkick(int N, const double* m, double* x, const double* v,
                    const oracle_params* p, double tau);

/* O9, reading G4: exact two-body propagation of one body about mu by dt,
 * eccentric / hyperbolic anomaly-difference form.  Returns 0, or -1 if the
 * root solve failed (never observed).                                        */
int oracle_kepler_drift_one(double mu, double dt, double x[3], double v[3]);
int oracle_drift(int N, double* x, double* v, const oracle_params* p, double dt);

/* O10: K(dt/2) S(dt/2) D(dt) S(dt/2) K(dt/2).                                */
int oracle_step(int N, const double* m, double* x, double* v,
                const oracle_params* p, double dt);

/* nsteps concatenated O10 steps with adjacent half-kicks merged:
 * K(dt/2) [S D S K(dt)]^(nsteps-1) S D S K(dt/2); r_crit is recomputed at each
 * force evaluation from the velocities of that moment (reading R7). */
int oracle_run(int N, const double* m, double* x, double* v,
               const oracle_params* p, double dt, int nsteps);

/* NEXT-1 (reading R11; GPU: params.encounter_mode = 1): the hybrid step with the encounter complement,
 * B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2), A = flow of Kepler + sum (1-K)-weighted pair terms integrated with
 * nsub RK4 substeps for all bodies (r_crit,ij held at the opening evaluation's values).  weight_mode must be 1. */
void oracle_encounter_drift(int N, const double* m, double* x, double* v, const oracle_params* p,
                            const double* rc, const double* sa, const double* vk, double dt, int nsub);
int oracle_step_hybrid(int N, const double* m, double* x, double* v, const oracle_params* p, double dt, int nsub);
/* the same step with A(dt) integrated by Gragg-Bulirsch-Stoer extrapolation to the relative tolerance tol (reading R15;
 * PAPER.md:45 names the integrator); stats (may be NULL): accepted macro steps, rejected, right-hand sides */
int oracle_encounter_drift_bs(int N, const double* m, double* x, double* v, const oracle_params* p,
                              const double* rc, const double* sa, const double* vk, double dt, double tol, long long* stats);
int oracle_step_hybrid_bs(int N, const double* m, double* x, double* v, const oracle_params* p, double dt, double tol,
                          long long* stats);
/* NEXT-3, reading R16: L levels of changeover with radius ratio F and S sub-steps per level; shell
 * weight of level l (0 <= l < L: W_l - W_{l-1}; l == L: the remainder 1 - W_{L-1} that Bulirsch-Stoer integrates) */
double oracle_level_weight(double r, double rcrit, int l, int L, double F);
int oracle_step_multilevel(int N, const double* m, double* x, double* v, const oracle_params* p, double dt,
                           int L, int S, double F, double tol, long long* stats);

/* O11.  E = sum m v^2/2 + |sum m v|^2/(2 M_star) - sum G M_star m/r
 *                         - sum_{i<j} G m_i m_j / r_ij ;  L = sum m x cross v. */
void oracle_energy_angmom(int N, const double* m, const double* x, const double* v,
                          const oracle_params* p, double* E, double L[3]);

/* NEXT-4 ("collisions ... perfect mergers"; reading R13): step-end collision pass.
 * Collision graph: i ~ j iff r_ij < R_i + R_j (strict; R = physical radii) at the given positions.  Every
 * connected component of more than one body becomes ONE body at the component's smallest index:
 * m = sum m_k, x = sum m_k x_k / m, v = sum m_k v_k / m (v: the stored democratic velocities, so
 * sum m v and sum m x are unchanged), R = cbrt(sum R_k^3); a component of total mass 0 keeps the x, v of
 * its smallest index.  The other members are removed and the arrays closed up in order.  Sums run
 * over the members in ascending index.  newidx[N] (may be NULL): the new index of each old body
 * (of its survivor, for a removed body).  Returns the new body count.                                */
int oracle_merge(int N, double* m, double* x, double* v, double* R, int* newidx);
/* TP2 mode (reading R9): only pairs with i < n_big or j < n_big exist; *n_big_new = big bodies left.             */
int oracle_merge_tp2(int N, double* m, double* x, double* v, double* R, int* newidx, int n_big, int* n_big_new);
/* Reading R14 (NOT built on the GPU yet): the hybrid step with the collision pass after every RK4 substep of the
 * A-flow; the merged body inherits the frozen r_crit,i, a_i, v_K,i of the component's smallest index.  Returns N'. */
int oracle_step_hybrid_collide(int N, double* m, double* x, double* v, double* R, const oracle_params* p,
                               double dt, int nsub, int* newidx);
int oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
