// genga_internal.cuh -- handle layout, workspace carving and kernel launchers shared by the
// translation units of libgenga_b200.  Product code: nothing here is used by oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/genga.h"

namespace genga {

// ---- tiling constants -------------------------------------------------
// j-bodies per chunk (granularity of the near-field flag and of the FP32 frames): a template parameter
// CHUNK of the kernels, 128 by default and 64 for small systems, where the (i-block, chunk) units are too
// few to spread evenly over the CTAs (Handle::chunk).
constexpr int CHUNK_MIN  = 64;
constexpr int CHUNK_MAX  = 128;
constexpr int STAGE_J    = 1024;                // j-bodies per shared-memory stage (STAGE_J / CHUNK chunks)
constexpr int NSTAGE     = 2;                   // double buffering
constexpr int PAD_BODIES = 512;                 // N is padded to a multiple of this (stage and i-block size)
constexpr double PAD_POS = 1.0e15;              // position of padding bodies (gm = 0, far from everything)

// per-body / per-chunk parameters of the conservative near-field bound (all FP32, rounded up):
//   B_ic = max( max(hq_i, Hq_c) * max(aq_i, Aq_c), max(rf_i, Rf_c) ),  bound_ic = B_ic^2
struct __align__(16) BoundP { float hq, aq, rf, pad; };

// per-chunk record staged next to the j-tile: the maxima of the bound parameters over the chunk
// and the origin of the chunk's local frame (FP32 policy P32: the FP32 kernel sees positions
// relative to o; Rf already contains the frame guard floor * 2 * max_j |x_j - o|).
struct __align__(16) ChunkP { double ox, oy, oz; float hq, aq, rf, rad; float q2max, uni; };   // uni = 1: every slot of the chunk is live and all carry bitwise the same G m (else 0)
static_assert(sizeof(ChunkP) == 48, "ChunkP is staged with 16-byte bulk copies");

// j-side layouts.  FP32: two bodies per pair of float4 (packed for FFMA2 along j), in two planes per chunk:
//   [CHUNK/2] float4 A = (x0, x1, y0, y1), then [CHUNK/2] float4 B = (z0, z1, gm0, gm1)
//   (lanes that read consecutive pairs hit consecutive 16-byte words: conflict-free LDS.128).
// FP64: double4 (x, y, z, gm) per body.
// FP32 positions are relative to the origin of the body's own chunk (ChunkP).
struct Counters {
    unsigned int cand_count;     // (body, chunk) candidates pushed by the all-pairs kernel
    unsigned int pair_count;     // encounter pairs appended by the near-field kernel
    unsigned int noconv;         // bodies whose Kepler solve did not converge (sticky until read)
    unsigned int overflow;       // 1 if the last near-field pass took the exact slow path
    unsigned int ticket;         // block-completion ticket of the momentum reduction (0 between launches)
    unsigned int extent_bits;    // float bits of max(|x|, |y|) over the bodies (Hilbert sort extent)
    // encounter mode (encounter.cuh; NEXT-1)
    unsigned int enc_status;     // sticky until read: 1 pair list overflowed, 2 a group had more than enc::GBIG bodies, 8 the Bulirsch-Stoer step size collapsed
    unsigned int enc_groups;     // encounter groups integrated by the last drift
    unsigned int enc_bodies;     // bodies in those groups
    unsigned int enc_maxsize;    // largest group of the last drift
    unsigned int enc_missed;     // sticky until read: pairs found inside their zone after a drift that had not grouped them
    unsigned int enc_merged;     // bodies absorbed by mergers inside the encounter integration since the last genga_merge (reading R14)
    unsigned int enc_rhs_sum;    // force evaluations of the group integrations of the last drift: all groups, ...
    unsigned int enc_rhs_max;    // ... the most any group needed (the drift waits for that group), ...
    unsigned int enc_rejected;   // ... and Bulirsch-Stoer macro steps that were rejected
    // mergers (merge.cu; NEXT-4): written by the last genga_merge
    unsigned int merge_n;        // body count after the pass
    unsigned int merge_status;   // 1 pair list had overflowed, 2 a radius exceeds half its critical radius
    unsigned int merge_nbig;     // TP2 mode: big bodies after the pass
};

struct Workspace {
    // state (API layout)
    double* m;        // [NP]
    double* x;        // [NP][3]
    double* v;        // [NP][3]
    double* a;        // [NP][3]  acceleration of the last force evaluation
    double* a2;       // [NP][3]  the other acceleration buffer of the small-system kernel (lean_step.cu); a and a2 change places
    // per-body derived
    double* hcbrt;    // [NP] cbrt(m / 3 M_star), cached when masses change
    double* rcrit;    // [NP]
    double* semi;     // [NP]
    double* vkep;     // [NP]
    // arrays of one force evaluation, in the INTERNAL (sorted) order: slot s holds body order[s]
    int*     order;   // [NP]   slot -> body index (API order); order[s] = s for the padding slots s >= N
    unsigned long long* keys;   // [NP] sort keys (heavy class, Hilbert index, body index)
    unsigned long long* bkeys;  // [NP] the keys grouped by bucket
    int* bigslot;               // [NP] TP2 mode: slot of big body b (b < n_big)
    unsigned int* sortbuf;      // bucket histogram, starts and cursors of the sort
    int* glabel;                // [2 NP] encounter mode: smallest body index of the body's encounter group (-1: none,
                                //        -2: group too large, Kepler drift), then [NP] member count / group index per label
    int* ginfo;                 // [2 x max groups] (offset, member count) per group, then the member lists (body indices)
    int* gulist;                // [min(2 pair_cap, NP)] the bodies that occur in the pair list, each once
    double4* pk64;    // [NP]   (x, y, z, G m)
    float4*  pk32;    // [NP]   two planes per chunk, see above
    double4* aux;     // [NP]   (m, r_crit, a, v_K): what the exact pair rule O3 needs
    BoundP*  bi;      // [NP]   per-body bound parameters
    ChunkP*  bc;      // [NP/chunk] per-chunk maxima and frame origin
    // lists
    int2*    cand;    // [cand_cap] (body, chunk)
    int2*    pairs;   // [pair_cap] (i, j), i < j
    // scratch
    double*  red;     // [RED_DOUBLES] reduction scratch / results
    double*  vtmp;    // [NP][3] staging for heliocentric-velocity output
    double*  mom;     // momentum slots and per-block partials of the fused step (momentum.cuh)
    double*  radius;  // [NP] physical radii R_i (genga_set_radii; 0 = the body never collides)
    int*     absorb;  // [NP] reading R14: body that absorbed this one inside an encounter integration (-1: none); genga_merge closes up
    double*  aslot;   // [3][NP] sums of the symmetric all-pairs kernels in the internal order (kick_sym_body.cuh: aslot_index),
                      //         zeroed by the prep step, folded into a[] by the near-field kernel
    unsigned long long* leanx;   // [LEANX_WORDS] exchange slots of the small-system kernel (lean_step.cu: exchange_sums); written by
                      //         nothing else, and only ever with growing sequence numbers (zero at genga_create)
    Counters* ctr;
};
constexpr int LEANX_WORDS = 8192;

constexpr int RED_DOUBLES = 8 + 8 * 1024;   // [0..7] results, [8..8+4096) pair-potential partials, then momentum partials

struct Handle {
    int N, NP, nchunk;
    int chunk;                   // CHUNK of this handle: 64 or 128
    genga_params p;
    double lambda_near, near_floor;
    int pair_cap, cand_cap;
    cudaStream_t stream;
    Workspace w;
    int num_sms;
    long long launches;
    // internal order (a performance hint only: results never depend on it)
    int mega_blocks[2];          // co-resident blocks of the one-kernel step per precision; 0 = not used, -1 = not queried yet
    int mega_nmax;               // largest N that takes the one-kernel step
    int lean_blocks[2];          // CTAs of the small-system kernel (lean_step.cu) per precision; 0 = not used, -1 = not queried yet
    int lean_nmax;               // largest N that takes it
    int lean_min_evals;          // ... and the shortest sequence of force evaluations that does
    unsigned long long lean_seq; // grid-wide exchanges its launches have done (the slots in w.mom carry the number, never cleared)
    int enc_blocks;              // co-resident grid of the per-body kernel built with the encounter integrator
    bool enc_labels_valid;       // glabel holds the groups of the drift that led to the current positions
    double enc_dt;               // |dt| of the drift the next listing is for (the last sequence's; params.dt_rcrit before any)
    int fused_blocks;            // co-resident blocks of the fused per-body kernel; 0 = cooperative launch unavailable
    bool pend_vel;               // a closing velocity update v += pend_tau a is still owed (api.cu: sequence)
    double pend_tau;
    bool mom_a_valid;            // mom[SLOT_A] holds sum m v of the stored velocities
    bool mom_b_valid;            // mom[SLOT_B] holds sum m v' of the last drift and only kicks have touched v since: by reading R17
                                 // it is the momentum the next Sun-kick needs (never set in TP2 mode: forces are not reciprocal there)
    bool pairs_current;          // the encounter list was made from the current positions (genga_merge relies on it)
    int grid_cache[2][2];        // per kernel (FP32, FP64): variant + 1 it was computed for, grid size
    int tune[4];                 // genga_set_tuning: [0] kick32 variant, [1] kick64 variant
    int resort_every;            // force evaluations between two sorts
    int evals_since_sort;        // < 0: no order yet

    // profiling
    int prof;
    static constexpr int NKT = 4;
    static constexpr int EVPOOL = 256;
    cudaEvent_t ev0[NKT][EVPOOL], ev1[NKT][EVPOOL];
    int evn[NKT];
    double ms_total[NKT];
    long long ms_launches[NKT];
    bool events_created;
};

size_t carve_workspace(int N, int pair_cap, int cand_cap, void* base, Workspace* w);

// ---- kernel launchers (each in its own .cu) ---------------------------------------------------
struct PrepArgs {
    int N, NP;
    double G, M_star, n1, n2, dt_rcrit;
    int pair_rule;
    int n_big;                   // TP2 mode (>= 0): prep also records the slots of the big bodies
    float lambda, floor_rel;     // near-field policy for this evaluation
    int scaled;                  // FP32 j-records in the mass-scaled form (kick_fp32.cu, SC variants)
    double preshift;             // pending Sun-kick: x += preshift * mom[SLOT_B] / M_star before anything else
};
struct EncArgs {                  // encounter mode (encounter.cuh; NEXT-1, reading R11)
    int on;                        // 0: every body drifts on its Kepler orbit
    int nsub;                      // > 0: RK4 with nsub substeps per step for the bodies of an encounter group; 0: Bulirsch-Stoer
    int pair_rule;
    unsigned int pair_cap;
    double G, M_star, n1, n2dt;
    double tol;                    // nsub <= 0: relative tolerance of the Bulirsch-Stoer integration (encounter.cuh)
    int levels, levels_sub;        // reading R16: changeover levels (1: the two-level step) and sub-steps per level
    double level_ratio;            // radius ratio between consecutive levels
    int collide;                   // RK4 only: collision pass after every substep (reading R14)
    int maxgroups;                 // layout of Workspace::ginfo: [2 maxgroups] (offset, count) per group, then the member lists
};
struct OnBodyArgs {               // the fused per-body kernel of the step (fused_step.cu)
    PrepArgs prep;
    EncArgs enc;
    int do_vel, do_drift, do_prep;
    int reuse_P;                   // do_drift: take sum m v from mom[SLOT_B] instead of summing it (reading R17)
    double tau_v;                  // v += tau_v a          (do_vel)
    double dt, mu;                 // S(dt/2) D(dt) S(dt/2)  (do_drift; the closing S is applied by phase 3)
};
constexpr int MOM_MAX_BLOCKS = 2048;   // most blocks whose momentum partials fit the workspace
int  onbody_max_blocks(const Handle* h, bool enc);
cudaError_t launch_groups(const Handle* h);                      // encounter groups from the pair list (encounter.cuh)
cudaError_t launch_onbody(const Handle* h, const OnBodyArgs& a, int max_blocks);
int  mega_max_blocks(const Handle* h, int precision);            // the one-kernel step of small systems (mega_step.cu)
cudaError_t launch_step_mega(const Handle* h, const OnBodyArgs& a, int precision, int max_blocks);
int  lean_max_blocks(const Handle* h, int precision);            // sequences of steps of a small system in one kernel (lean_step.cu)
int  lean_nmax_limit();
cudaError_t launch_lean(const Handle* h, const PrepArgs& prep, int precision, int lead, int n_sds, int pend,
                        double tau_prev, double tau_first, double tau_mid, double dt, int max_blocks,
                        unsigned long long seq0);                 // leaves a in w.a2; seq0: grid-wide exchanges done so far
void launch_hcbrt(const Handle* h);
void launch_pad(const Handle* h);                            // padding bodies: x = (PAD_POS,0,0), v = 0, m = 0
int  sort_buffer_words();
void launch_sort(const Handle* h);                           // order[] by (heavy class, semi-major axis)
void launch_prep(const Handle* h, const PrepArgs& a);
void launch_kick32(const Handle* h);
void launch_kick64(const Handle* h);
void launch_nearfield(const Handle* h);
void launch_tp2(const Handle* h);                            // TP2 mode: big bodies against all (FP64)
void launch_momentum(const Handle* h);                       // red[0..2] = sum m v, red[3] = sum m
void launch_momentum_slot_a(const Handle* h);                // the same into mom[SLOT_A]
void launch_velupdate_mom(const Handle* h, double tau);      // v += tau a; mom[SLOT_A] = sum m v
void launch_shift_drift_mom(const Handle* h, double tau_pre, double dt);   // S(tau_pre) D(dt); mom[SLOT_B] = sum m v
void launch_shift_v(const Handle* h, double scale);          // v_i += scale * red[0..2]   (O1)
void launch_sunkick(const Handle* h, double tau);            // x_i += tau * red[0..2] / M_star
void launch_drift(const Handle* h, double dt);
void launch_merge(const Handle* h, int* newidx_dev);            // step-end perfect mergers (merge.cu, reading R13)
void launch_energy(const Handle* h);                         // red[0] = E, red[1..3] = L
void launch_copy_v_helio(const Handle* h, const double* mom, double* out);   // out = v + mom[0..2]/M_star
int  run_peak_probe(int which, int iters, cudaStream_t s, double* ops_per_s, double* ms);

// occupancy-derived grid of the all-pairs kernels
int kick32_grid(const Handle* h);
int kick64_grid(const Handle* h);
int kick32_num_variants();
bool kick32_variant_scaled(int v);      // does this variant read mass-scaled j-records?
int kick64_num_variants();
const char* kick32_variant_name(int v);
const char* kick64_variant_name(int v);

}  // namespace genga
