/*
 * genga.h -- C ABI of libgenga_b200: the level-0 hot path of the GENGA hybrid symplectic
 * N-body step (arXiv 2309.08217) as hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Citations: PAPER.md:NN = line NN of the paper text; G1..G12 / O1..O11 are the readings and
 * oracle steps of SURVEY.md section 8(c), restated in DESIGN.md section 3.
 *
 * What is computed
 *   kick: a_i = sum_{j != i} G m_j K(r_ij, r_crit,ij) (x_j - x_i)/r_ij^3,
 *        K the changeover function (reading G1), r_crit,i from Eq. 1,
 *        in FP64 or FP32 force precision ("Do Kick in single precision");
 *        pairs with r_ij < r_crit,ij are recorded as close-encounter candidates.
 *   drift ("the Kepler orbit solver is always performed in double precision"):
 *        exact two-body propagation about mu = G M_star with universal-variable f and g.
 *   step  (reading G3): K(dt/2) S(dt/2) D(dt) S(dt/2) K(dt/2) in democratic
 *        heliocentric variables (heliocentric x, barycentric v).
 *   energy_angmom: total energy E and angular momentum L of the stored state.
 *   merge ("perfect mergers"; reading R13, optional): overlapping bodies (r_ij < R_i + R_j) become one
 *        at a step end; N shrinks.  genga_set_radii / genga_merge / genga_num_bodies / genga_get_mass below.
 *
 * Conventions
 *   N        number of bodies, the star excluded.  N = 0 and N = 1 are valid.  N only changes in genga_merge.
 *   m        [N]      FP64 masses.  m = 0 (test particle) is valid.
 *   x, v, a  [N][3]   FP64, row-major (a contiguous (N,3) float64 tensor).  x is heliocentric.
 *            The STORED velocity is barycentric ("democratic").  If params.v_is_heliocentric,
 *            genga_create / genga_set_state convert the velocities they are given (O1).
 *   DEVICE   pointer into CUDA device memory of the current device.
 *   HOST     pointer into host memory (pinned memory makes the copies asynchronous).
 *   Every call except the ones marked "synchronises" only enqueues work on params.stream.
 *   The library never allocates device memory: all state lives in params.workspace, owned by the
 *   caller (size from genga_workspace_bytes) and must stay valid until genga_destroy.
 *   Input pointers are borrowed for the duration of the call (DEVICE inputs: until the enqueued
 *   copy has run, i.e. stream order).  One handle is not thread-safe; handles share no state.
 *   Return value: GENGA_OK (0) or a negative genga_status.  No exceptions, no abort.
 *
 *   The workspace layout is private: read the state only through the accessors below.  (The closing
 *   velocity update of genga_kick/step/run/leapfrog is deferred into the first kernel of the next such
 *   call and is applied by any accessor or state-changing call that comes first.)
 *
 * There is NO CPU fallback: without a CUDA device every compute call returns GENGA_ECUDA.
 */
#ifndef GENGA_H
#define GENGA_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct genga_s* genga_handle;

typedef enum {
    GENGA_OK        =  0,
    GENGA_EINVAL    = -1,   /* bad argument (NULL handle, N < 0, unknown precision, ...)            */
    GENGA_ENOMEM    = -2,   /* params.workspace_bytes < genga_workspace_bytes(N, params)            */
    GENGA_ECAPACITY = -3,   /* encounter-pair list overflow: first cap pairs written, *count = total */
    GENGA_ECUDA     = -4,   /* a CUDA runtime call failed; genga_last_cuda_error() has the text      */
    GENGA_ENOCONV   = -5,   /* Kepler solver failed to converge for >= 1 body (state still written)  */
    GENGA_ELIMIT    = -6    /* size beyond the fixed maximum of a no-allocation entry point          */
} genga_status;

/* PAPER.md:223 "Do Kick in single precision = 0 / 1". */
typedef enum { GENGA_FP64 = 0, GENGA_FP32 = 1 } genga_precision;

/* Reading G2: how r_crit,ij follows from per-body quantities.
 *   PAIR_MAX         r_crit,ij = max(r_crit,i, r_crit,j)                      (Eq. 1 per body)
 *   PAIR_MUTUAL_HILL r_crit,ij = max(n1 ((m_i+m_j)/(3 M_star))^(1/3) (a_i+a_j)/2,
 *                                    n2 dt_rcrit max(v_K,i, v_K,j))           (BASELINE configs) */
typedef enum { GENGA_PAIR_MAX = 0, GENGA_PAIR_MUTUAL_HILL = 1 } genga_pair_rule;

typedef struct {
    double G;                 /* gravitational constant in the caller's units (k^2 for AU, day, Msun)  */
    double M_star;            /* central mass                                                          */
    double n1, n2;            /* Eq. 1 (3 and 0.4; BASELINE configs: 3 and 0)              */
    double dt_rcrit;          /* the dt of Eq. 1's second term (reading G8: the step dt)               */
    int    pair_rule;         /* genga_pair_rule                                                       */
    int    v_is_heliocentric; /* 1: velocities given to create/set_state are heliocentric (O1)         */
    double lambda_near;       /* FP32 policy P32: pairs with r_ij < lambda_near * r_crit,ij (as bounded
                                 per j-chunk) are evaluated in FP64.  <= 0 selects the default (2).    */
    double near_floor;        /* FP32 policy P32: the FP32 kernel sees positions relative to the origin
                                 of each j-chunk (params.chunk bodies); every pair with r_ij < near_floor * 2 R_chunk
                                 (R_chunk = radius of the chunk about its origin) is evaluated in FP64
                                 (position-rounding guard: relative separation error <= 2^-24 / near_floor).
                                 < 0 selects the default (1/256); 0 disables.                           */
    void*  stream;            /* cudaStream_t owned by the caller; NULL = the legacy default stream    */
    void*  workspace;         /* DEVICE memory owned by the caller, 256-byte aligned                    */
    size_t workspace_bytes;
    int    pair_capacity;     /* capacity (pairs) of the encounter-pair list kept inside the workspace */
    int    cand_capacity;     /* capacity of the internal (body, j-chunk) near-field candidate list;
                                 <= 0 selects a default.  Overflow is handled exactly (slow path).      */
    int    resort_every;      /* force evaluations between two refreshes of the internal body order
                                 (heavy bodies first, then along a Hilbert curve in the x-y plane; a
                                 performance hint only).  <= 0: default (8; 32 if N < 16384).              */
    int    chunk;             /* j-bodies per chunk (granularity of the near flag and of the FP32 frames): 64 or
                                 128; anything else selects the default per force evaluation (64 below N = 14 000
                                 with FP32 forces and below N = 20 000 with FP64 forces, else 128)            */
    int    mega_nmax;         /* systems of up to this many bodies run a whole force evaluation (per-body
                                 kernel, all-pairs kick, near field) as ONE cooperative kernel (7 % faster at
                                 N <= 2048, slower from N = 4096 on); 0: default (3000), < 0: never                                                              */
    int    lean_nmax;         /* systems of up to this many bodies run whole SEQUENCES of force evaluations and steps
                                 (genga_kick/step/run/leapfrog) in one kernel in which every CTA holds the whole
                                 system in shared memory and only the pair sums are shared out: one grid-wide
                                 barrier per step instead of three launches (csrc/lean_step.cu; not in TP2 or
                                 encounter mode, not while profiling).  0: default (2560, the most an SM's
                                 shared memory holds at 80 bytes per body), < 0: never                     */
    int    lean_min_evals;    /* ... and only for sequences of at least this many force evaluations: a launch
                                 of that kernel first loads the whole system into every CTA (~11 us at
                                 N = 1024), which a single genga_step does not win back.  0: default (4)  */
    int    n_big;             /* TP2 mode ("the giant planets feel the forces of the planetesimals,
                                 but the planetesimals do not feel each other"; reading R9): a pair
                                 (i, j) interacts iff i < n_big or j < n_big.  < 0 (default): every pair.
                                 The O(n_big N) pair sums of this mode always run in FP64.              */
    int    weight_mode;       /* pair weight inside a changeover zone (reading R10): 0 (default) W = K,
                                 as north_star words it; 1: W = K - r dK/dr, the gradient of the pair
                                 potential -G m_i m_j K / r (Hamiltonian-consistent level-0 kick)       */
    int    no_fused_step;     /* 1: genga_kick/step/run/leapfrog use the separate per-body kernels instead of the
                                 one cooperative kernel per step (debugging; also taken if the device lacks
                                 cooperative launch)                                                   */
    int    encounter_mode;    /* NEXT-1 (reading R11), opt-in.  0 (default): every body
                                 moves on its Kepler orbit during the drift (the level-0 step of north_star).
                                 1: the hybrid symplectic step: the bodies of an
                                 encounter GROUP (connected component of the encounter-pair list of the step's
                                 opening force evaluation) are advanced over dt under their Kepler terms plus the
                                 complement pair forces G m_j (1 - (K - r dK/dr)) / r^2, in FP64, by Bulirsch-Stoer
                                 extrapolation to enc_tol (or enc_nsub RK4 substeps), r_crit,ij held at the opening
                                 evaluation's values.  Groups of up to 16 bodies take a warp, up to 256 a CTA; larger
                                 ones are dissolved (their bodies drift on Kepler orbits) and reported (status bit 2).
                                 Requires weight_mode = 1, n_big < 0 and the cooperative per-body kernel.    */
    int    enc_nsub;          /* > 0: the groups are integrated with classical RK4, enc_nsub equal substeps per step (the scheme of
                                 oracle_step_hybrid); <= 0 (default): Gragg-Bulirsch-Stoer extrapolation to enc_tol            */
    double enc_list_scale;    /* encounter mode: which pairs OUTSIDE their zone are listed (and grouped) as well, so that
                                 a pair that enters its zone DURING the step is already in a group: those with
                                 r_ij < enc_list_scale * r_crit,ij  and  r_ij - r_crit,ij < enc_list_vfactor * dt * |v_i - v_j|
                                 (dt: the step of the running genga_step/run/leapfrog call; params.dt_rcrit before the
                                 first).  1 <= enc_list_scale <= 8, <= 0: default (8).  Changes the list
                                 genga_encounter_pairs returns, not the forces.  Pairs that got into their zone
                                 un-grouped all the same are counted (genga_encounter_stats).                       */
    double enc_list_vfactor;  /* see enc_list_scale.  0: default (1.25); < 0: no velocity test, every pair inside
                                 enc_list_scale * r_crit,ij is listed.                                               */
    double enc_tol;           /* encounter mode, enc_nsub <= 0: relative tolerance of the Bulirsch-Stoer integration of the groups
                                 (reading R15): a macro step is accepted when the last extrapolation
                                 correction of every member is below enc_tol in |dx|/|x| and |dv|/|v|; <= 0: default 1e-12.
                                 genga_encounter_stats status bit 8: the step size collapsed (dt 2^-30) without convergence  */
    int    enc_collide;       /* reading R14 ("collisions ... perfect mergers"), opt-in; needs encounter_mode = 1 and
                                 enc_nsub > 0 (else GENGA_EINVAL).  1: after every RK4 substep of a group's integration its
                                 members are tested for r_kl < R_k + R_l (genga_set_radii) and every connected component of
                                 overlapping bodies becomes one body at its smallest index on the spot (m, centre of mass,
                                 momentum and sum R^3 kept; the merged body keeps the frozen r_crit,i, a_i, v_K,i of that
                                 index), which is how bodies that pass through each other WITHIN a step are caught.  The
                                 absorbed bodies stay in the arrays as massless bodies of radius -1e300 until the next
                                 genga_merge closes the arrays up (its newidx and n_merged account for them).            */
    int    enc_levels;        /* NEXT-3, reading R16 ("levels" and "sub-steps"): number of changeover levels of
                                 the encounter integration; <= 1 (default): the two-level step (level 0 + Bulirsch-Stoer).
                                 L > 1 (<= 4; needs encounter_mode = 1 and enc_nsub <= 0): level l = 1 .. L - 1 is a symplectic
                                 kick-flow-kick with the step dt / enc_substeps^l on the shell
                                 (W(r; r_crit / F^l) - W(r; r_crit / F^(l-1))) of the pair potential, F = enc_level_ratio,
                                 and Bulirsch-Stoer integrates the Kepler terms plus the innermost remainder
                                 1 - W(r; r_crit / F^(L-1)) over dt / enc_substeps^(L-1).                                 */
    int    enc_substeps;      /* sub-steps per level; <= 0: default 3                                                     */
    double enc_level_ratio;   /* radius ratio F > 1 between consecutive levels; 0: default enc_substeps^(2/3) (Kepler scaling) */
} genga_params;

/* Fill *p with the defaults: G = k^2 (k = 0.01720209895), M_star = 1, n1 = 3, n2 = 0,
 * dt_rcrit = 0, PAIR_MUTUAL_HILL, v_is_heliocentric = 1, lambda_near/near_floor = defaults,
 * stream/workspace = NULL, capacities = defaults.                                             */
void   genga_default_params(genga_params* p);

/* Bytes of DEVICE workspace a handle for N bodies needs with these params (capacities resolved). */
size_t genga_workspace_bytes(int N, const genga_params* p);

/* Create a handle; copies m, x, v (DEVICE pointers, [N], [N][3], [N][3]) into the workspace on
 * params.stream.  m/x/v may be NULL (state zero-initialised; use genga_set_state* later).      */
int genga_create(genga_handle* out, int N, const double* m, const double* x, const double* v,
                 const genga_params* p);
int genga_destroy(genga_handle h);

/* Replace the state.  DEVICE pointers / HOST pointers.  Any of m, x, v may be NULL (kept).      */
int genga_set_state(genga_handle h, const double* m, const double* x, const double* v);
int genga_set_state_host(genga_handle h, const double* m, const double* x, const double* v);

/* Kick: r_crit (Eq. 1), force evaluation in the given precision, encounter-pair list, and
 * v_i += dt * a_i with exactly the dt given (dt < 0 allowed).  PAPER.md:43, 55, 223.            */
int genga_kick(genga_handle h, double dt, int precision);

/* Refresh the internal body order now (it is refreshed automatically at the first force
 * evaluation and then every params.resort_every evaluations).                                  */
int genga_resort(genga_handle h);

/* Force evaluation only (as genga_kick with the velocity update left out).                      */
int genga_accel(genga_handle h, int precision);

/* Kepler drift only: every body propagated by dt about mu = G M_star (O9).         */
int genga_drift(genga_handle h, double dt);

/* Sun-kick only: x_i += tau * (sum_j m_j v_j) / M_star (reading G3; O8).                        */
int genga_sunkick(genga_handle h, double tau);

/* One step K(dt/2) S(dt/2) D(dt) S(dt/2) K(dt/2) (O10): two force evaluations.                  */
int genga_step(genga_handle h, double dt, int precision);

/* nsteps steps with adjacent half-kicks merged: K(dt/2) [S D S K(dt)]^(nsteps-1) S D S K(dt/2),
 * nsteps + 1 force evaluations (reading R7).                                          */
int genga_run(genga_handle h, double dt, int nsteps, int precision);
/* (genga_run and genga_leapfrog hand systems of up to params.lean_nmax bodies to one kernel for the whole
 * sequence: issue the steps of a run in one call rather than one by one.  Inside such a call the momentum of
 * the Sun-kick before a drift is the one summed after the previous drift, reading R17, and the
 * sums of the few pairs inside their near bound are added in no fixed order: the accelerations of bodies
 * with two or more such pairs are reproducible to rounding, not bit for bit.)                            */

/* The body of that loop on its own: [S(dt/2) D(dt) S(dt/2) K(dt)]^nsteps, one force evaluation
 * per step.  genga_kick(dt/2), genga_leapfrog(n), genga_kick(-dt/2) equals genga_run(n) up to
 * rounding as long as no pair sits inside a changeover zone (r_crit depends on v through a_i).   */
int genga_leapfrog(genga_handle h, double dt, int nsteps, int precision);

/* Encounter pairs {(i,j): i < j, r_ij < r_crit,ij} of the LAST force evaluation.
 * pairs_ij: HOST int[cap][2] (may be NULL if cap = 0); *count (HOST) receives the true total.
 * Order unspecified.  Synchronises the stream.                                                  */
int genga_encounter_pairs(genga_handle h, int* pairs_ij, int cap, int* count);

/* E and L of the stored state (O11).  HOST outputs.  Synchronises the stream.     */
int genga_energy_angmom(genga_handle h, double* E, double L[3]);

/* Accessors.  DEVICE outputs (asynchronous) and HOST outputs (synchronise).  NULL = skip.
 * x heliocentric; v as stored (barycentric) unless heliocentric_v != 0 (O1 inverse).            */
int genga_get_state(genga_handle h, double* x, double* v, int heliocentric_v);
int genga_get_state_host(genga_handle h, double* x, double* v, int heliocentric_v);
int genga_get_accel(genga_handle h, double* a);          /* DEVICE [N][3]: a_i of the last force evaluation.  The a_i are
                                                             sums of per-(body, chunk) partials added with FP64 atomics
                                                             in no fixed order (all-pairs kernels, near field, merged
                                                             states in genga_merge): equal from run to run to rounding
                                                             (1e-16 relative), not bit for bit.  The momentum sums of
                                                             the step are combined in a fixed order.                   */
int genga_get_rcrit(genga_handle h, double* rcrit);      /* DEVICE [N]: r_crit,i of the last force evaluation */

/* ---- perfect mergers at a step end (NEXT-4; "collisions ... perfect mergers"; R13) ----
 * genga_set_radii: physical radii R_i, DEVICE double[N] borrowed for the call (NULL: all 0 = no body ever
 * collides, the state after genga_create).  genga_get_radii: DEVICE double[N] output.  Asynchronous.
 *
 * genga_merge: bodies i, j collide iff r_ij < R_i + R_j (strict, FP64) at the current positions.  Every
 * connected component of the collision graph becomes ONE body at the component's smallest index:
 * m = sum m_k, x = sum m_k x_k / m, v = sum m_k v_k / m (stored velocities: total momentum and the centre of
 * mass are kept), R = cbrt(sum R_k^3); a component of total mass 0 keeps its first member's x, v.  The other
 * members are removed and m, x, v, R closed up IN ORDER: afterwards the handle holds N' = N - *n_merged
 * bodies (genga_num_bodies) and every accessor uses N'.  The workspace is not re-carved.
 *   Candidates are the pairs of the encounter list of the last force evaluation, so R_i + R_j <= r_crit,ij is
 * required (status bit 2 is raised if some 2 R_i > r_crit,i); if the positions have changed since that
 * evaluation (genga_drift, genga_sunkick, genga_set_state) one is run first, in `precision`; when bodies were
 * merged, one is run afterwards, so that the pair list, a_i and r_crit,i describe the new body set.
 *   newidx: DEVICE int[N] (N before the call) or NULL: new index of each old body (of the body that absorbed
 * it).  n_merged, status: HOST outputs (NULL = skip); status bit 1: the pair list had overflowed (pairs may
 * have been missed).  Synchronises the stream.
 *   TP2 mode (params.n_big): only pairs with a big body exist, so small bodies never merge with each other; the
 * handle's n_big becomes the number of survivors among the big bodies (genga_num_big_bodies).                  */
int genga_set_radii(genga_handle h, const double* R);
int genga_get_radii(genga_handle h, double* R);
int genga_get_mass(genga_handle h, double* m);           /* DEVICE double[N]: the masses (they change with mergers) */
int genga_merge(genga_handle h, int precision, int* newidx, int* n_merged, int* status);
int genga_num_bodies(genga_handle h);                    /* current N (shrinks with mergers); < 0 on a NULL handle */
int genga_num_big_bodies(genga_handle h);                /* current params.n_big (-1: every pair interacts, or NULL) */

/* Diagnostics of the last force evaluation: number of (body, j-chunk) near-field candidates and
 * whether the candidate list overflowed (exact slow path taken).  HOST outputs.  Synchronises.  */
int genga_nearfield_stats(genga_handle h, long long* candidates, int* overflowed);

/* Encounter mode: the groups the last drift integrated (their number, the bodies in them, the largest), the
 * number of pairs that a force evaluation found INSIDE their zone (r_ij < r_crit,ij) although the drift that led
 * there had not moved them as one group (they entered un-grouped: raise enc_list_scale or shorten dt), and a
 * status mask; count and mask are cleared by this call.  Mask: 1 the pair list overflowed when the groups were
 * formed (raise pair_capacity), 2 a group had more than 8 bodies (its bodies drifted on their Kepler orbits
 * instead), 4 missed_pairs > 0, 8 the adaptive substep hit its floor (an approach too deep to resolve: raise enc_nsub).
 * HOST outputs, NULL = skip.  Synchronises.  GENGA_EINVAL unless
 * params.encounter_mode = 1.                                                                          */
int genga_encounter_stats(genga_handle h, int* groups, int* bodies, int* largest, int* missed_pairs, int* status);

/* Encounter mode: the work of the group integrations of the LAST drift: force evaluations
 * summed over all groups, the most any one group needed (the drift waits for that group) and the Bulirsch-Stoer
 * macro steps that were rejected.  HOST pointers (any may be NULL); synchronises.  GENGA_EINVAL outside encounter mode. */
int genga_encounter_work(genga_handle h, long long* rhs_total, int* rhs_max, int* rejected);

/* Per-kernel device timing.  enable is a bit mask: bit k brackets every launch of kernel class k with
 * CUDA events on params.stream; classes: 0 all-pairs kick kernel, 1 near-field kernel, 2 prep kernel,
 * 3 drift kernel (15 = all, 0 = off).  genga_kernel_time returns, for class which, the summed
 * milliseconds and launch count since the last reset (HOST outputs).  Synchronises.              */
int genga_set_profiling(genga_handle h, int enable);
int genga_kernel_time(genga_handle h, int which, double* ms_total, long long* launches, int reset);

/* Kernel configuration ("tuning", cf. GENGA's self-tuning): key 0 selects the
 * launch/tiling variant of the FP32 all-pairs kernel, key 1 of the FP64 one; value in
 * [0, genga_num_variants(key)); 0 is the default.  Keys 2 (FP32) and 3 (FP64) set the grid of that kernel in
 * half waves of co-resident CTAs, 1..64; 0 (default): up to four waves with at least 16 j-chunks per CTA.
 * Results are identical up to summation order.  GENGA_EINVAL for any other key or value.           */
int genga_set_tuning(genga_handle h, int key, int value);
/* Time every variant of the given precision's all-pairs kernel on the current state (force evaluation
 * = prep + all-pairs + near field, 1 warm-up + 3 timed runs each) and keep the fastest.  HOST
 * outputs (may be NULL): the chosen variant and its time.  The stored state is unchanged; the
 * acceleration and pair list are those of the last timed evaluation.  Synchronises.               */
int genga_autotune(genga_handle h, int precision, int* chosen, double* ms_best);
int genga_num_variants(int key);
const char* genga_variant_name(int key, int value);

/* Launches issued by this handle since creation (kernels only, not copies).                     */
long long genga_launch_count(genga_handle h);

int genga_synchronize(genga_handle h);
const char* genga_strerror(int code);
const char* genga_last_cuda_error(void);
const char* genga_version(void);

/* ALU peak probes: run a register-only dependent-chain kernel on every SM
 * for iters iterations and return achieved instr throughput.  which: 0 FFMA, 1 FFMA2 (packed),
 * 2 DFMA, 3 MUFU.RSQ, 4 MUFU.RSQ64H (anything else: GENGA_EINVAL).  *ops_per_s (HOST) = lane-operations
 * per second (an FFMA2 counts 2).  stream as in params.  Synchronises.  bench.py prints these beside the
 * derived peaks its roofline fractions are quoted against.                                              */
int genga_peak_probe(int which, int iters, void* stream, double* ops_per_s, double* ms);

/* ---- an entry point that allocates nothing ---------------------------------------------------------------
 * E and L (O11) of a state given as plain DEVICE arrays, for callers that cannot allocate (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): no handle, no workspace.
 * Its scratch (the bodies packed into padded tiles, the per-block partials of the pair potential) is a
 * file-scope __device__ array of the library (csrc/noalloc.cu), 4.2 MB that every GPU holds from the moment
 * it loads the library until the process exits.  The call makes no cudaMalloc / cudaFree and calls no
 * allocating library routine; the first call on a device asks the runtime for the array's device address.
 *   N      bodies, 0 <= N <= GENGA_STATIC_NMAX; more: GENGA_ELIMIT (text: genga_static_last_error())
 *   m      DEVICE double[N]; x, v: DEVICE double[N][3], x heliocentric, v barycentric (democratic variables:
 *          what genga_get_state returns with heliocentric_v = 0)
 *   G, M_star   as in genga_params (M_star > 0)
 *   stream cudaStream_t (NULL: the default stream) of the CURRENT device; the arrays must live there
 *   out4   DEVICE double[4], receives (E, Lx, Ly, Lz); written asynchronously on `stream`
 * Same arithmetic as genga_energy_angmom (every pair interacts: no TP2 case); the results agree to rounding
 * (the summation order of the pair potential follows the padding: 128 here, 512 there).
 * ALL calls share the one array, which keeps the last call's contents (nothing in it needs clearing: a call
 * rewrites all it reads): calls on one stream are ordered and safe, calls that OVERLAP on the GPU (different
 * streams or unordered host threads) race on it and return garbage.  Asynchronous; nothing is synchronised. */
#define GENGA_STATIC_NMAX 131072
int genga_energy_angmom_static(int N, const double* m, const double* x, const double* v, double G, double M_star,
                               void* stream, double* out4);
/* Text of the last error of genga_energy_angmom_static in this host thread ("" if none).                    */
const char* genga_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GENGA_H */
