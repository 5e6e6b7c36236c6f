// api.cu -- the C ABI of include/genga.h: argument checking, workspace carving, stream order of
// the kernels, host<->device copies, per-kernel event timing.  No arithmetic of the method lives
// here; every step of the path runs in the CUDA kernels of this directory.
#include "genga_internal.cuh"

#include <cmath>
#include <cstdio>
#include <algorithm>
#include <cstring>
#include <new>

namespace genga {

static thread_local char g_cuda_err[256] = "";

static int cuda_fail(cudaError_t e, const char* where)
{
    std::snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", where, cudaGetErrorString(e));
    return GENGA_ECUDA;
}
#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, #call); } while (0)
#define LAUNCHED(h, name) do { ++(h)->launches; cudaError_t e_ = cudaGetLastError(); \
                               if (e_ != cudaSuccess) return cuda_fail(e_, name); } while (0)

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

static int padded(int N) { return (int)align_up((size_t)(N > 0 ? N : 1), PAD_BODIES); }

static void resolve_caps(int N, const genga_params* p, int* pair_cap, int* cand_cap)
{
    long long pc = p->pair_capacity > 0 ? p->pair_capacity : (4LL * N + 1024);
    long long cc = p->cand_capacity > 0 ? p->cand_capacity : (16LL * N + 65536);
    if (pc > 0x3fffffff) pc = 0x3fffffff;
    if (cc > 0x3fffffff) cc = 0x3fffffff;
    *pair_cap = (int)pc; *cand_cap = (int)cc;
}

size_t carve_workspace(int N, int pair_cap, int cand_cap, void* base, Workspace* w)
{
    const size_t NP = (size_t)padded(N);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    const size_t o_m = take(NP * 8), o_x = take(NP * 24), o_v = take(NP * 24), o_a = take(NP * 24);
    const size_t o_h = take(NP * 8), o_rc = take(NP * 8), o_sa = take(NP * 8), o_vk = take(NP * 8);
    const size_t o_p64 = take(NP * 32), o_p32 = take(NP * 16), o_bi = take(NP * 16), o_bc = take(NP / CHUNK_MIN * sizeof(ChunkP));
    const size_t o_cand = take((size_t)cand_cap * 8), o_pairs = take((size_t)pair_cap * 8);
    const size_t o_red = take((size_t)RED_DOUBLES * 8), o_vt = take(NP * 24), o_ctr = take(sizeof(Counters));
    const size_t o_ord = take(NP * 4), o_key = take(NP * 8), o_aux = take(NP * 32);
    const size_t o_mom = take((8 + 4 * (NP / 128 + 1) + 8 * (size_t)MOM_MAX_BLOCKS) * 8);
    const size_t o_bs = take(NP * 4);
    const size_t o_bk = take(NP * 8), o_sb = take((size_t)sort_buffer_words() * 4);
    const size_t o_gl = take(NP * 8);          // labels [NP], member counts [NP]
    const size_t o_gi = take(std::min((size_t)pair_cap, NP / 2) * 9 * 4);      // encounter groups: count + 8 members each
    const size_t o_gu = take(std::min(2 * (size_t)pair_cap, NP) * 4);
    const size_t o_rad = take(NP * 8);
    const size_t o_as = take(NP * 24);
    const size_t o_ab = take(NP * 4);
    const size_t o_a2 = take(NP * 24);
    const size_t o_lx = take((size_t)LEANX_WORDS * 8);
    if (w && base) {
        char* b = static_cast<char*>(base);
        w->m = (double*)(b + o_m); w->x = (double*)(b + o_x); w->v = (double*)(b + o_v); w->a = (double*)(b + o_a);
        w->hcbrt = (double*)(b + o_h); w->rcrit = (double*)(b + o_rc); w->semi = (double*)(b + o_sa);
        w->vkep = (double*)(b + o_vk); w->pk64 = (double4*)(b + o_p64); w->pk32 = (float4*)(b + o_p32);
        w->bi = (BoundP*)(b + o_bi); w->bc = (ChunkP*)(b + o_bc); w->cand = (int2*)(b + o_cand);
        w->pairs = (int2*)(b + o_pairs); w->red = (double*)(b + o_red); w->vtmp = (double*)(b + o_vt);
        w->ctr = (Counters*)(b + o_ctr);
        w->order = (int*)(b + o_ord); w->keys = (unsigned long long*)(b + o_key); w->aux = (double4*)(b + o_aux);
        w->mom = (double*)(b + o_mom);
        w->bigslot = (int*)(b + o_bs);
        w->bkeys = (unsigned long long*)(b + o_bk); w->sortbuf = (unsigned int*)(b + o_sb);
        w->glabel = (int*)(b + o_gl); w->ginfo = (int*)(b + o_gi); w->gulist = (int*)(b + o_gu);
        w->radius = (double*)(b + o_rad);
        w->aslot = (double*)(b + o_as);
        w->absorb = (int*)(b + o_ab);
        w->a2 = (double*)(b + o_a2);
        w->leanx = (unsigned long long*)(b + o_lx);
    }
    return off;
}

// ---- profiling -------------------------------------------------------------------------------
static int prof_flush(Handle* h, int which)
{
    for (int k = 0; k < h->evn[which]; ++k) {
        CU(cudaEventSynchronize(h->ev1[which][k]));
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, h->ev0[which][k], h->ev1[which][k]));
        h->ms_total[which] += ms;
        ++h->ms_launches[which];
    }
    h->evn[which] = 0;
    return GENGA_OK;
}

struct ProfScope {
    Handle* h; int which; bool on;
    ProfScope(Handle* h_, int w_) : h(h_), which(w_), on(((h_->prof >> w_) & 1) != 0)
    {
        if (!on) return;
        if (h->evn[which] == Handle::EVPOOL) prof_flush(h, which);
        cudaEventRecord(h->ev0[which][h->evn[which]], h->stream);
    }
    ~ProfScope()
    {
        if (!on) return;
        cudaEventRecord(h->ev1[which][h->evn[which]], h->stream);
        ++h->evn[which];
    }
};

// Refresh the internal order (heavy bodies first, then by semi-major axis).
static int resort(Handle* h)
{
    if (h->N == 0) return GENGA_OK;
    launch_momentum(h); LAUNCHED(h, "momentum_kernel");     // red[3] = sum m (mean mass -> heavy class)
    launch_sort(h); h->launches += 5;
    { cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) return cuda_fail(e_, "sort kernels"); }
    h->evals_since_sort = 0;
    return GENGA_OK;
}

// ---- force evaluation -------------------------------------------------------------------------
// Chunk size of the next force evaluation: 128, or 64 for smaller systems (more tiles to spread over the warps).  The
// symmetric FP64 kernel keeps gaining from 64-body chunks up to N ~ 20 000 (N = 16 384: 223 against 240 us), the FP32 one
// up to ~14 000 (N = 16 384: 123 against 116 us).  params.chunk overrides.  Everything that depends on the chunk size
// (packing, frames, bounds, candidate list) is rebuilt by every evaluation, so it may change from one to the next.
static void set_chunk(Handle* h, int precision)
{
    int c = h->p.chunk;
    if (c != CHUNK_MIN && c != CHUNK_MAX) c = (h->N < (precision == GENGA_FP64 ? 20000 : 14000)) ? CHUNK_MIN : CHUNK_MAX;
    if (c != h->chunk) { h->chunk = c; h->grid_cache[0][0] = h->grid_cache[1][0] = 0; }
    h->nchunk = (h->N + h->chunk - 1) / h->chunk;      // j-chunks that hold a live body (pure padding is skipped)
}

static int maybe_resort(Handle* h)
{
    if (h->evals_since_sort < 0 || h->evals_since_sort >= h->resort_every) {
        const int rc = resort(h);
        if (rc != GENGA_OK) return rc;
    }
    ++h->evals_since_sort;
    return GENGA_OK;
}

static PrepArgs make_prep_args(const Handle* h, int precision, double preshift)
{
    PrepArgs a;
    a.N = h->N; a.NP = h->NP;
    a.G = h->p.G; a.M_star = h->p.M_star; a.n1 = h->p.n1; a.n2 = h->p.n2; a.dt_rcrit = h->p.dt_rcrit;
    a.pair_rule = h->p.pair_rule;
    a.n_big = (h->p.n_big >= 0 && h->p.n_big < h->N) ? h->p.n_big : -1;
    a.preshift = preshift;
    a.scaled = (precision == GENGA_FP32 && kick32_variant_scaled(h->tune[0])) ? 1 : 0;
    if (precision == GENGA_FP32) {
        a.lambda = (float)h->lambda_near;
        // never below 2^-18: closer pairs have no meaning in FP32 (and mass-scaled self/coincident residues stay flagged)
        a.floor_rel = (float)(h->near_floor > 3.814697265625e-06 ? h->near_floor : 3.814697265625e-06);
    }
    else                         { a.lambda = 1.0f;                  a.floor_rel = 0.0f; }
    // encounter mode lists (and must therefore look at) every pair within enc_list_scale r_crit
    if (h->p.encounter_mode == 1 && a.lambda < (float)h->p.enc_list_scale) a.lambda = (float)h->p.enc_list_scale;
    return a;
}

// all-pairs kernel + near-field kernel on the arrays the prep step packed
static int launch_pairs(Handle* h, int precision)
{
    if (h->p.n_big >= 0 && h->p.n_big < h->N) {          // TP2 mode: O(n_big N) pairs, FP64 (reading R9)
        if (h->p.n_big > 0) { ProfScope ps(h, 0); launch_tp2(h); LAUNCHED(h, "tp2_kernel"); }
        h->pairs_current = h->p.n_big > 0;              // only a kernel that rebuilt the list makes it current
        return GENGA_OK;
    }
    { ProfScope ps(h, 0); if (precision == GENGA_FP32) launch_kick32(h); else launch_kick64(h); }
    LAUNCHED(h, "kick_kernel");
    { ProfScope ps(h, 1); launch_nearfield(h); }
    LAUNCHED(h, "nearfield_kernel");
    h->pairs_current = true;
    return GENGA_OK;
}

static int force_eval(Handle* h, int precision, double preshift = 0.0)
{
    if (precision != GENGA_FP64 && precision != GENGA_FP32) return GENGA_EINVAL;
    if (h->N == 0) return GENGA_OK;
    set_chunk(h, precision);
    const int rc = maybe_resort(h);
    if (rc != GENGA_OK) return rc;
    const PrepArgs a = make_prep_args(h, precision, preshift);
    { ProfScope ps(h, 2); launch_prep(h, a); }
    LAUNCHED(h, "prep_kernel");
    return launch_pairs(h, precision);
}

// The fused per-body kernel (fused_step.cu): [v += tau_v a] [S(dt/2) D(dt)] [S(dt/2), r_crit, pack].
static int onbody(Handle* h, int precision, bool do_vel, double tau_v, bool do_drift, double dt, bool do_prep)
{
    if (h->N == 0) return GENGA_OK;
    OnBodyArgs a;
    if (do_prep) {
        set_chunk(h, precision);
        const int rc = maybe_resort(h);
        if (rc != GENGA_OK) return rc;
    }
    a.prep = make_prep_args(h, precision, 0.0);
    a.do_vel = do_vel; a.do_drift = do_drift; a.do_prep = do_prep;
    a.tau_v = tau_v; a.dt = dt; a.mu = h->p.G * h->p.M_star;
    const bool enc = h->p.encounter_mode == 1 && do_drift;
    // (not with encounter groups: their warps read velocities that other blocks have just updated, which the barrier of the sum orders)
    a.reuse_P = (do_drift && h->mom_b_valid && !enc) ? 1 : 0;
    a.enc.on = enc ? 1 : 0; a.enc.nsub = h->p.enc_nsub; a.enc.pair_rule = h->p.pair_rule;
    a.enc.pair_cap = (unsigned int)h->pair_cap;
    a.enc.G = h->p.G; a.enc.M_star = h->p.M_star; a.enc.n1 = h->p.n1; a.enc.n2dt = h->p.n2 * h->p.dt_rcrit;
    a.enc.tol = h->p.enc_tol;
    a.enc.collide = h->p.enc_collide;
    a.enc.levels = h->p.enc_levels; a.enc.levels_sub = h->p.enc_substeps; a.enc.level_ratio = h->p.enc_level_ratio;
    a.enc.maxgroups = (int)std::min((size_t)h->pair_cap, (size_t)h->NP / 2);
    cudaError_t e;
    if (enc) {                                         // groups of the pair list the last force evaluation left
        if (!h->pairs_current) {                       // no list of the current positions (first call after create /
            const int rc = force_eval(h, precision);   // set_state / genga_drift / genga_sunkick): make one, or the
            if (rc != GENGA_OK) return rc;             // complement forces of the pairs inside their zones are lost
            a.prep = make_prep_args(h, precision, 0.0);
        }
        e = launch_groups(h);
        ++h->launches;
        if (e != cudaSuccess) return cuda_fail(e, "group_kernel");
        h->enc_labels_valid = true;
    }
    { ProfScope ps(h, do_drift ? 3 : 2); e = launch_onbody(h, a, (enc && h->enc_blocks < h->fused_blocks) ? h->enc_blocks : h->fused_blocks); }
    ++h->launches;
    if (e != cudaSuccess) return cuda_fail(e, "onbody_kernel (cooperative launch)");
    h->mom_a_valid = !do_drift;          // slot A holds sum m v of the stored velocities unless the drift changed them
    if (do_drift) h->mom_b_valid = !(h->p.n_big >= 0 && h->p.n_big < h->N);   // slot B: sum m v' (reading R17; not in TP2 mode)
    return GENGA_OK;
}

static int to_democratic(Handle* h)
{
    if (h->N == 0) return GENGA_OK;
    launch_momentum(h); LAUNCHED(h, "momentum_kernel");
    launch_shift_v(h, -1.0); LAUNCHED(h, "shift_kernel");
    return GENGA_OK;
}

}  // namespace genga

using namespace genga;

struct genga_s : public genga::Handle {};

// K(tau): force evaluation, v += tau a, and (fused) the momentum of the new velocities.  preshift:
// a pending Sun-kick S(preshift) with the momentum the fused drift left in mom[SLOT_B].
static int kick_fused(genga_handle h, double tau, int precision, double preshift)
{
    const int rc = force_eval(h, precision, preshift);
    if (rc != GENGA_OK) return rc;
    if (h->N == 0) return GENGA_OK;
    launch_velupdate_mom(h, tau); LAUNCHED(h, "velupdate_mom_kernel");
    h->mom_a_valid = true;
    return GENGA_OK;
}

// S(dt/2) D(dt) of one step in ONE kernel (reading G3); the closing S(dt/2) is left pending for the
// prep kernel of the kick that always follows inside genga_step / genga_run / genga_leapfrog.
static int sd_fused(genga_handle h, double dt)
{
    if (h->N == 0) return GENGA_OK;
    if (!h->mom_a_valid) { launch_momentum_slot_a(h); LAUNCHED(h, "momentum_kernel"); }
    { ProfScope ps(h, 3); launch_shift_drift_mom(h, 0.5 * dt, dt); }
    LAUNCHED(h, "shift_drift_mom_kernel");
    h->mom_a_valid = false;
    return GENGA_OK;
}

// The one-kernel step of small systems (mega_step.cu): usable for this call?
static bool mega_ready(Handle* h, int precision)
{
    if (h->fused_blocks <= 0 || h->prof != 0 || h->N > h->mega_nmax) return false;
    if (h->p.n_big >= 0 && h->p.n_big < h->N) return false;          // TP2 mode has its own pair kernel
    if (h->p.encounter_mode == 1) return false;                      // the groups are formed between two launches
    const int pi = precision == GENGA_FP32 ? 1 : 0;
    if (h->mega_blocks[pi] < 0) h->mega_blocks[pi] = mega_max_blocks(h, precision);
    return h->mega_blocks[pi] > 0;
}

// [v += tau_v a] [S(dt/2) D(dt)] S(dt/2), r_crit, pack, all-pairs kick, near field: one cooperative launch.
static int step_mega(Handle* h, int precision, bool do_vel, double tau_v, bool do_drift, double dt)
{
    set_chunk(h, precision);
    const int rc = maybe_resort(h);
    if (rc != GENGA_OK) return rc;
    OnBodyArgs a;
    std::memset(&a.enc, 0, sizeof(a.enc));
    a.prep = make_prep_args(h, precision, 0.0);
    a.prep.scaled = 0;                                               // the fused all-pairs phase reads plain j-records
    a.do_vel = do_vel; a.do_drift = do_drift; a.do_prep = 1;
    a.tau_v = tau_v; a.dt = dt; a.mu = h->p.G * h->p.M_star;
    a.reuse_P = (do_drift && h->mom_b_valid) ? 1 : 0;
    const cudaError_t e = launch_step_mega(h, a, precision, h->mega_blocks[precision == GENGA_FP32 ? 1 : 0]);
    ++h->launches;
    if (e != cudaSuccess) return cuda_fail(e, "step_kernel (cooperative launch)");
    h->pairs_current = true;
    h->mom_a_valid = !do_drift;
    if (do_drift) h->mom_b_valid = true;                             // (mega_ready excludes TP2 mode)
    return GENGA_OK;
}

// The small-system kernel (lean_step.cu): usable for this call?
static bool lean_ready(Handle* h, int precision)
{
    if (h->fused_blocks <= 0 || h->prof != 0 || h->N > h->lean_nmax) return false;
    if (h->p.n_big >= 0 && h->p.n_big < h->N) return false;          // TP2 mode has its own pair kernel
    if (h->p.encounter_mode == 1) return false;                      // the groups are formed between two launches
    const int pi = precision == GENGA_FP32 ? 1 : 0;
    if (h->lean_blocks[pi] < 0) h->lean_blocks[pi] = lean_max_blocks(h, precision);
    return h->lean_blocks[pi] > 0;
}

// The sequence of sequence() below in as few launches of the small-system kernel as the re-sorts allow: the
// order may only change between two launches.  pending / tau_prev: the velocity update still owed on entry.
static int sequence_lean(Handle* h, int precision, bool lead_kick, double tau_first, int n_sds, double dt,
                         double tau_mid, bool pending, double tau_prev)
{
    const int E = (lead_kick ? 1 : 0) + n_sds;
    int e0 = 0;
    while (e0 < E) {
        if (h->evals_since_sort < 0 || h->evals_since_sort >= h->resort_every) {
            const int rc = resort(h);
            if (rc != GENGA_OK) return rc;
        }
        int c = h->resort_every - h->evals_since_sort;
        if (c > E - e0) c = E - e0;
        if (c > 4096) c = 4096;                                      // one launch should not hold the device for much longer than a second
        const int lead = (lead_kick && e0 == 0) ? 1 : 0;
        const bool pend = e0 == 0 ? pending : true;
        const double tp = e0 == 0 ? tau_prev : ((lead_kick && e0 == 1) ? tau_first : tau_mid);
        const PrepArgs a = make_prep_args(h, precision, 0.0);
        const cudaError_t e = launch_lean(h, a, precision, lead, c - lead, pend ? 1 : 0, tp, tau_first, tau_mid, dt,
                                          h->lean_blocks[precision == GENGA_FP32 ? 1 : 0], h->lean_seq);
        h->lean_seq += 2ull * (unsigned long long)(c - lead) + 1ull;  // two exchanges per step (+ one a lone kick may do)
        ++h->launches;
        if (e != cudaSuccess) return cuda_fail(e, "lean_kernel (cooperative launch)");
        std::swap(h->w.a, h->w.a2);                                   // the kernel leaves the new accelerations in the other buffer
        h->evals_since_sort += c;
        e0 += c;
    }
    h->pairs_current = true;
    return GENGA_OK;
}

// K(tau_first)? then n_sds times [S(dt/2) D(dt) S(dt/2) K(tau)], tau = tau_mid except tau_last for the last
// one.  Fused path: one per-body kernel between two force evaluations (3 launches per step).
static int sequence(genga_handle h, int precision, bool lead_kick, double tau_first, int n_sds, double dt,
                    double tau_mid, double tau_last)
{
    if (precision != GENGA_FP64 && precision != GENGA_FP32) return GENGA_EINVAL;
    int rc;
    if (h->N == 0) return GENGA_OK;
    if (h->fused_blocks <= 0) {                                     // no cooperative launch: the un-fused kernels
        if (h->pend_vel) return GENGA_EINVAL;                       // cannot happen: only the fused path defers
        if (lead_kick && (rc = kick_fused(h, tau_first, precision, 0.0)) != GENGA_OK) return rc;
        for (int k = 0; k < n_sds; ++k) {
            if ((rc = sd_fused(h, dt)) != GENGA_OK) return rc;
            if ((rc = kick_fused(h, k == n_sds - 1 ? tau_last : tau_mid, precision, 0.5 * dt)) != GENGA_OK) return rc;
        }
        return GENGA_OK;
    }
    // The closing velocity update of a sequence is DEFERRED (h->pend_vel): it rides in the first per-body
    // kernel of the next sequence, or is flushed by the first call that reads or replaces the state.
    bool pending = h->pend_vel;
    double tau_prev = h->pend_tau;
    h->pend_vel = false;
    if (n_sds > 0) h->enc_dt = std::fabs(dt);                        // encounter mode: the listings of this sequence look dt ahead
    if ((lead_kick ? 1 : 0) + n_sds >= h->lean_min_evals && lean_ready(h, precision)) {   // small system: the whole sequence in one kernel
        if ((rc = sequence_lean(h, precision, lead_kick, tau_first, n_sds, dt, tau_mid, pending, tau_prev)) != GENGA_OK) return rc;
        h->pend_vel = true; h->pend_tau = n_sds > 0 ? tau_last : tau_first; h->mom_a_valid = false;
        if (n_sds > 0) h->mom_b_valid = true;                        // the kernel's last drift left sum m v' in slot B
        return GENGA_OK;
    }
    const bool mega = mega_ready(h, precision);                      // small system: one launch per force evaluation
    if (lead_kick) {
        if (mega) { if ((rc = step_mega(h, precision, pending, tau_prev, false, 0.0)) != GENGA_OK) return rc; }
        else {
            if ((rc = onbody(h, precision, pending, tau_prev, false, 0.0, true)) != GENGA_OK) return rc;
            if ((rc = launch_pairs(h, precision)) != GENGA_OK) return rc;
        }
        pending = true; tau_prev = tau_first;
    }
    for (int k = 0; k < n_sds; ++k) {
        if (mega) { if ((rc = step_mega(h, precision, pending, tau_prev, true, dt)) != GENGA_OK) return rc; }
        else {
            if ((rc = onbody(h, precision, pending, tau_prev, true, dt, true)) != GENGA_OK) return rc;
            if ((rc = launch_pairs(h, precision)) != GENGA_OK) return rc;
        }
        pending = true; tau_prev = (k == n_sds - 1) ? tau_last : tau_mid;
    }
    if (pending) { h->pend_vel = true; h->pend_tau = tau_prev; h->mom_a_valid = false; }
    return GENGA_OK;
}

// Apply a deferred velocity update (see sequence()).  Called by everything that reads or replaces x, v.
static int flush_pending(genga_handle h)
{
    if (!h->pend_vel) return GENGA_OK;
    h->pend_vel = false;
    if (h->N == 0) return GENGA_OK;
    // one plain kernel: v += tau a and, in its epilogue, sum m v of the new velocities (slot A), which a read of the
    // heliocentric velocities needs next; the cooperative per-body kernel would cost three times as much here
    launch_velupdate_mom(h, h->pend_tau); LAUNCHED(h, "velupdate_mom_kernel");
    h->mom_a_valid = true;
    return GENGA_OK;
}

extern "C" {

void genga_default_params(genga_params* p)
{
    if (!p) return;
    std::memset(p, 0, sizeof(*p));
    p->G = 0.01720209895 * 0.01720209895;
    p->M_star = 1.0;
    p->n1 = 3.0; p->n2 = 0.0; p->dt_rcrit = 0.0;
    p->pair_rule = GENGA_PAIR_MUTUAL_HILL;
    p->v_is_heliocentric = 1;
    p->lambda_near = 0.0; p->near_floor = -1.0;
    p->stream = nullptr; p->workspace = nullptr; p->workspace_bytes = 0;
    p->pair_capacity = 0; p->cand_capacity = 0;
    p->resort_every = 0;
    p->no_fused_step = 0;
    p->n_big = -1;
    p->chunk = 0;
    p->mega_nmax = 0;
    p->lean_nmax = 0;
    p->lean_min_evals = 0;
    p->weight_mode = 0;
    p->encounter_mode = 0; p->enc_nsub = 0; p->enc_list_scale = 0.0; p->enc_list_vfactor = 0.0; p->enc_tol = 0.0; p->enc_collide = 0; p->enc_levels = 0; p->enc_substeps = 0; p->enc_level_ratio = 0.0;
}

size_t genga_workspace_bytes(int N, const genga_params* p)
{
    if (N < 0 || !p) return 0;
    int pc, cc;
    resolve_caps(N, p, &pc, &cc);
    return carve_workspace(N, pc, cc, nullptr, nullptr);
}

int genga_create(genga_handle* out, int N, const double* m, const double* x, const double* v, const genga_params* p)
{
    if (!out || !p || N < 0 || N > (1 << 20)) return GENGA_EINVAL;
    if (!(p->M_star > 0.0) || !(p->G > 0.0)) return GENGA_EINVAL;
    if (p->pair_rule != GENGA_PAIR_MAX && p->pair_rule != GENGA_PAIR_MUTUAL_HILL) return GENGA_EINVAL;
    if (p->weight_mode != 0 && p->weight_mode != 1) return GENGA_EINVAL;
    if (p->encounter_mode != 0 && p->encounter_mode != 1) return GENGA_EINVAL;
    if (p->encounter_mode == 1 && (p->weight_mode != 1 || (p->n_big >= 0 && p->n_big < N) || p->no_fused_step)) return GENGA_EINVAL;
    if (p->enc_collide != 0 && (p->enc_collide != 1 || p->encounter_mode != 1 || p->enc_nsub <= 0)) return GENGA_EINVAL;
    if (p->enc_levels > 1 && (p->encounter_mode != 1 || p->enc_nsub > 0 || p->enc_levels > 4 || p->enc_substeps < 0 ||
                              (p->enc_level_ratio != 0.0 && !(p->enc_level_ratio > 1.0)))) return GENGA_EINVAL;
    *out = nullptr;
    int pc, cc;
    resolve_caps(N, p, &pc, &cc);
    const size_t need = carve_workspace(N, pc, cc, nullptr, nullptr);
    if (!p->workspace || p->workspace_bytes < need) return GENGA_ENOMEM;
    if ((reinterpret_cast<uintptr_t>(p->workspace) & 255u) != 0) return GENGA_EINVAL;

    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));

    genga_s* h = new (std::nothrow) genga_s();
    if (!h) return GENGA_ENOMEM;
    std::memset(static_cast<Handle*>(h), 0, sizeof(Handle));
    h->N = N; h->NP = padded(N);
    // chunk size until the first force evaluation chooses its own (set_chunk)
    h->chunk = (p->chunk == CHUNK_MIN || p->chunk == CHUNK_MAX) ? p->chunk : (N < 14000 ? CHUNK_MIN : CHUNK_MAX);
    h->nchunk = (N + h->chunk - 1) / h->chunk;      // j-chunks that hold a live body (pure padding is skipped)
    h->p = *p;
    h->lambda_near = p->lambda_near > 0.0 ? p->lambda_near : 2.0;
    h->near_floor  = p->near_floor >= 0.0 ? p->near_floor : (1.0 / 256.0);
    if (h->lambda_near < 1.0) h->lambda_near = 1.0;
    h->pair_cap = pc; h->cand_cap = cc;
    // default: every 8 force evaluations where the all-pairs kernel dominates, every 32 for small systems
    // (the refresh is five tiny kernels, ~25 us, which a 40 us step should not pay too often)
    const bool tp2 = p->n_big >= 0 && p->n_big < N;             // O(n_big N) pairs: the order hardly matters
    h->resort_every = p->resort_every > 0 ? p->resort_every : (tp2 ? 64 : (N >= 16384 ? 8 : (N <= 4096 ? 128 : 32)));
    h->evals_since_sort = -1;
    h->stream = static_cast<cudaStream_t>(p->stream);
    h->num_sms = sms;
    {
        int coop = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        h->fused_blocks = (coop && !p->no_fused_step) ? onbody_max_blocks(h, false) : 0;
        if (p->encounter_mode == 1) {
            if (!coop) { delete h; return GENGA_EINVAL; }
            h->enc_blocks = onbody_max_blocks(h, true);
            h->p.enc_nsub = p->enc_nsub > 0 ? p->enc_nsub : 0;                 // 0: Bulirsch-Stoer to enc_tol
            h->p.enc_list_scale = p->enc_list_scale > 0.0 ? p->enc_list_scale : 8.0;
            h->p.enc_list_vfactor = p->enc_list_vfactor == 0.0 ? 1.25 : p->enc_list_vfactor;
            h->enc_dt = std::fabs(p->dt_rcrit);
            h->p.enc_tol = p->enc_tol > 0.0 ? p->enc_tol : 1.0e-12;
            h->p.enc_levels = p->enc_levels > 1 ? p->enc_levels : 1;
            h->p.enc_substeps = p->enc_substeps > 0 ? p->enc_substeps : 3;
            h->p.enc_level_ratio = p->enc_level_ratio > 1.0 ? p->enc_level_ratio : std::cbrt((double)h->p.enc_substeps * h->p.enc_substeps);
            if (h->p.enc_list_scale < 1.0 || h->p.enc_list_scale > 8.0) { delete h; return GENGA_EINVAL; }
        }
        h->mega_blocks[0] = h->mega_blocks[1] = -1;
        h->lean_blocks[0] = h->lean_blocks[1] = -1;
        h->lean_seq = 0;
        h->lean_min_evals = p->lean_min_evals > 0 ? p->lean_min_evals : 4;
        h->lean_nmax = p->lean_nmax > 0 ? std::min(p->lean_nmax, lean_nmax_limit()) : (p->lean_nmax < 0 ? 0 : lean_nmax_limit());
        h->mega_nmax = p->mega_nmax > 0 ? p->mega_nmax : (p->mega_nmax < 0 ? 0 : 3000);
    }
    carve_workspace(N, pc, cc, p->workspace, &h->w);

    cudaError_t e = cudaMemsetAsync(p->workspace, 0, need, h->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->w.absorb, 0xff, (size_t)h->NP * sizeof(int), h->stream);   // -1: nobody absorbed
    if (e != cudaSuccess) { delete h; return cuda_fail(e, "cudaMemsetAsync(workspace)"); }
    launch_pad(h);
    ++h->launches;
    *out = h;
    const int rc = genga_set_state(h, m, x, v);
    if (rc != GENGA_OK) { delete h; *out = nullptr; return rc; }
    return GENGA_OK;
}

int genga_destroy(genga_handle h)
{
    if (!h) return GENGA_EINVAL;
    if (h->events_created) {
        for (int w = 0; w < Handle::NKT; ++w)
            for (int k = 0; k < Handle::EVPOOL; ++k) { cudaEventDestroy(h->ev0[w][k]); cudaEventDestroy(h->ev1[w][k]); }
    }
    delete h;
    return GENGA_OK;
}

static int set_state_impl(genga_handle h, const double* m, const double* x, const double* v, cudaMemcpyKind kind)
{
    if (!h) return GENGA_EINVAL;
    if (v) h->pend_vel = false;                       // the owed update only touches v, which is replaced anyway
    { const int rcf = flush_pending(h); if (rcf != GENGA_OK) return rcf; }
    const size_t n = (size_t)h->N;
    if (n == 0) return GENGA_OK;
    if (m) CU(cudaMemcpyAsync(h->w.m, m, n * 8, kind, h->stream));
    if (x) { CU(cudaMemcpyAsync(h->w.x, x, n * 24, kind, h->stream)); h->enc_labels_valid = false; h->pairs_current = false; }
    if (v) { CU(cudaMemcpyAsync(h->w.v, v, n * 24, kind, h->stream)); h->mom_a_valid = false; h->mom_b_valid = false; }
    if (m) { h->mom_a_valid = false; h->mom_b_valid = false; h->pairs_current = false; h->enc_labels_valid = false; }   // r_crit follows m
    if (m) { launch_hcbrt(h); LAUNCHED(h, "hcbrt_kernel"); }
    if (v && h->p.v_is_heliocentric) return to_democratic(h);
    return GENGA_OK;
}

int genga_set_state(genga_handle h, const double* m, const double* x, const double* v)
{
    return set_state_impl(h, m, x, v, cudaMemcpyDeviceToDevice);
}

int genga_set_state_host(genga_handle h, const double* m, const double* x, const double* v)
{
    return set_state_impl(h, m, x, v, cudaMemcpyHostToDevice);
}

int genga_set_radii(genga_handle h, const double* R)
{
    if (!h) return GENGA_EINVAL;
    if (h->N == 0) return GENGA_OK;
    if (R) CU(cudaMemcpyAsync(h->w.radius, R, (size_t)h->N * 8, cudaMemcpyDeviceToDevice, h->stream));
    else   CU(cudaMemsetAsync(h->w.radius, 0, (size_t)h->N * 8, h->stream));
    return GENGA_OK;
}

int genga_get_radii(genga_handle h, double* R)
{
    if (!h || !R) return GENGA_EINVAL;
    if (h->N) CU(cudaMemcpyAsync(R, h->w.radius, (size_t)h->N * 8, cudaMemcpyDeviceToDevice, h->stream));
    return GENGA_OK;
}

int genga_get_mass(genga_handle h, double* m)
{
    if (!h || !m) return GENGA_EINVAL;
    if (h->N) CU(cudaMemcpyAsync(m, h->w.m, (size_t)h->N * 8, cudaMemcpyDeviceToDevice, h->stream));
    return GENGA_OK;
}

int genga_num_bodies(genga_handle h)
{
    return h ? h->N : GENGA_EINVAL;
}

int genga_num_big_bodies(genga_handle h)
{
    return h ? h->p.n_big : GENGA_EINVAL;
}

int genga_merge(genga_handle h, int precision, int* newidx, int* n_merged, int* status)
{
    if (!h || (precision != GENGA_FP64 && precision != GENGA_FP32)) return GENGA_EINVAL;
    if (n_merged) *n_merged = 0;
    if (status) *status = 0;
    if (h->N == 0) return GENGA_OK;
    int rc = flush_pending(h);
    if (rc != GENGA_OK) return rc;
    if (!h->pairs_current && (rc = force_eval(h, precision)) != GENGA_OK) return rc;
    launch_merge(h, newidx); h->launches += 2;
    { cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) return cuda_fail(e_, "merge kernels"); }
    h->enc_labels_valid = false;                                      // the label arrays served as scratch
    const bool tp2 = h->p.n_big >= 0 && h->p.n_big < h->N;
    unsigned int out[3];
    CU(cudaMemcpyAsync(out, &h->w.ctr->merge_n, sizeof(out), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    if (status) *status = (int)out[1];
    const int n_new = (int)out[0];
    if (n_new < 0 || n_new > h->N) return GENGA_ECUDA;
    if (n_merged) *n_merged = h->N - n_new;
    if (n_new == h->N) return GENGA_OK;
    // fewer bodies: the arrays keep their places in the workspace, everything derived from N is redone
    h->N = n_new; h->NP = padded(n_new);
    if (tp2) h->p.n_big = (int)out[2];                                 // merged big bodies leave one big body
    h->nchunk = (n_new + h->chunk - 1) / h->chunk;
    h->grid_cache[0][0] = h->grid_cache[1][0] = 0;
    h->evals_since_sort = -1;
    h->mom_a_valid = false;
    h->mom_b_valid = false;
    launch_pad(h); LAUNCHED(h, "pad_kernel");
    launch_hcbrt(h); LAUNCHED(h, "hcbrt_kernel");
    return force_eval(h, precision);                                  // pair list, a, r_crit of the new body set
}

int genga_resort(genga_handle h)
{
    if (!h) return GENGA_EINVAL;
    { const int rcf = flush_pending(h); if (rcf != GENGA_OK) return rcf; }
    return resort(h);
}

int genga_accel(genga_handle h, int precision)
{
    if (!h) return GENGA_EINVAL;
    { const int rcf = flush_pending(h); if (rcf != GENGA_OK) return rcf; }
    return force_eval(h, precision);
}

int genga_kick(genga_handle h, double dt, int precision)
{
    if (!h) return GENGA_EINVAL;
    return sequence(h, precision, true, dt, 0, 0.0, 0.0, 0.0);
}

int genga_drift(genga_handle h, double dt)
{
    if (!h) return GENGA_EINVAL;
    { const int rcf = flush_pending(h); if (rcf != GENGA_OK) return rcf; }
    { ProfScope ps(h, 3); launch_drift(h, dt); }
    LAUNCHED(h, "drift_kernel");
    h->pairs_current = false;
    h->mom_a_valid = false;
    h->mom_b_valid = false;
    h->enc_labels_valid = false;                     // a plain Kepler drift: no groups led to these positions
    return GENGA_OK;
}

int genga_sunkick(genga_handle h, double tau)
{
    if (!h) return GENGA_EINVAL;
    { const int rcf = flush_pending(h); if (rcf != GENGA_OK) return rcf; }
    if (h->N == 0) return GENGA_OK;
    launch_momentum(h); LAUNCHED(h, "momentum_kernel");
    launch_sunkick(h, tau); LAUNCHED(h, "sunkick_kernel");
    h->pairs_current = false;
    return GENGA_OK;
}

int genga_step(genga_handle h, double dt, int precision)
{
    if (!h) return GENGA_EINVAL;
    return sequence(h, precision, true, 0.5 * dt, 1, dt, 0.5 * dt, 0.5 * dt);
}

int genga_leapfrog(genga_handle h, double dt, int nsteps, int precision)
{
    if (!h || nsteps < 0) return GENGA_EINVAL;
    if (nsteps == 0) return GENGA_OK;
    return sequence(h, precision, false, 0.0, nsteps, dt, dt, dt);
}

int genga_run(genga_handle h, double dt, int nsteps, int precision)
{
    if (!h || nsteps < 0) return GENGA_EINVAL;
    if (nsteps == 0) return GENGA_OK;
    return sequence(h, precision, true, 0.5 * dt, nsteps, dt, dt, 0.5 * dt);
}

int genga_encounter_pairs(genga_handle h, int* pairs_ij, int cap, int* count)
{
    if (!h || !count || cap < 0 || (cap > 0 && !pairs_ij)) return GENGA_EINVAL;
    *count = 0;
    if (h->N == 0) return GENGA_OK;
    Counters c;
    CU(cudaMemcpyAsync(&c, h->w.ctr, sizeof(c), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    *count = (int)c.pair_count;
    unsigned int have = c.pair_count < (unsigned int)h->pair_cap ? c.pair_count : (unsigned int)h->pair_cap;
    unsigned int ncopy = have < (unsigned int)cap ? have : (unsigned int)cap;
    if (ncopy) {
        CU(cudaMemcpyAsync(pairs_ij, h->w.pairs, (size_t)ncopy * 8, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    return (c.pair_count > ncopy) ? GENGA_ECAPACITY : GENGA_OK;
}

int genga_energy_angmom(genga_handle h, double* E, double L[3])
{
    if (!h || !E || !L) return GENGA_EINVAL;
    { const int rcf = flush_pending(h); if (rcf != GENGA_OK) return rcf; }
    launch_energy(h); h->launches += 2;
    { cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) return cuda_fail(e_, "energy kernels"); }
    double r[4];
    CU(cudaMemcpyAsync(r, h->w.red, sizeof(r), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    *E = r[0]; L[0] = r[1]; L[1] = r[2]; L[2] = r[3];
    return GENGA_OK;
}

static int get_state_impl(genga_handle h, double* x, double* v, int helio, cudaMemcpyKind kind)
{
    if (!h) return GENGA_EINVAL;
    { const int rcf = flush_pending(h); if (rcf != GENGA_OK) return rcf; }
    const size_t n = (size_t)h->N;
    if (n == 0) return GENGA_OK;
    if (x) CU(cudaMemcpyAsync(x, h->w.x, n * 24, kind, h->stream));
    if (v) {
        if (helio) {
            const double* mom = h->w.mom;                      // slot A: sum m v of the stored velocities, if current
            if (!h->mom_a_valid) { launch_momentum(h); LAUNCHED(h, "momentum_kernel"); mom = h->w.red; }
            if (kind == cudaMemcpyDeviceToDevice) { launch_copy_v_helio(h, mom, v); LAUNCHED(h, "copy_shift_kernel"); }
            else {
                launch_copy_v_helio(h, mom, h->w.vtmp); LAUNCHED(h, "copy_shift_kernel");
                CU(cudaMemcpyAsync(v, h->w.vtmp, n * 24, kind, h->stream));
            }
        } else {
            CU(cudaMemcpyAsync(v, h->w.v, n * 24, kind, h->stream));
        }
    }
    if (kind == cudaMemcpyDeviceToHost) CU(cudaStreamSynchronize(h->stream));
    return GENGA_OK;
}

int genga_get_state(genga_handle h, double* x, double* v, int heliocentric_v)
{
    return get_state_impl(h, x, v, heliocentric_v, cudaMemcpyDeviceToDevice);
}

int genga_get_state_host(genga_handle h, double* x, double* v, int heliocentric_v)
{
    return get_state_impl(h, x, v, heliocentric_v, cudaMemcpyDeviceToHost);
}

int genga_get_accel(genga_handle h, double* a)
{
    if (!h || !a) return GENGA_EINVAL;
    if (h->N) CU(cudaMemcpyAsync(a, h->w.a, (size_t)h->N * 24, cudaMemcpyDeviceToDevice, h->stream));
    return GENGA_OK;
}

int genga_get_rcrit(genga_handle h, double* rcrit)
{
    if (!h || !rcrit) return GENGA_EINVAL;
    if (h->N) CU(cudaMemcpyAsync(rcrit, h->w.rcrit, (size_t)h->N * 8, cudaMemcpyDeviceToDevice, h->stream));
    return GENGA_OK;
}

int genga_nearfield_stats(genga_handle h, long long* candidates, int* overflowed)
{
    if (!h) return GENGA_EINVAL;
    Counters c;
    std::memset(&c, 0, sizeof(c));
    if (h->N) {
        CU(cudaMemcpyAsync(&c, h->w.ctr, sizeof(c), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    if (candidates) *candidates = (long long)c.cand_count;
    if (overflowed) *overflowed = (int)c.overflow;
    if (c.noconv) {                                   // sticky until reported once
        CU(cudaMemsetAsync(&h->w.ctr->noconv, 0, sizeof(unsigned int), h->stream));
        return GENGA_ENOCONV;
    }
    return GENGA_OK;
}

int genga_encounter_stats(genga_handle h, int* groups, int* bodies, int* largest, int* missed_pairs, int* status)
{
    if (!h || h->p.encounter_mode != 1) return GENGA_EINVAL;
    Counters c;
    std::memset(&c, 0, sizeof(c));
    if (h->N) {
        CU(cudaMemcpyAsync(&c, h->w.ctr, sizeof(c), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
        if (c.enc_missed) c.enc_status |= 4u;
        if (c.enc_status) CU(cudaMemsetAsync(&h->w.ctr->enc_status, 0, sizeof(unsigned int), h->stream));
        if (c.enc_missed) CU(cudaMemsetAsync(&h->w.ctr->enc_missed, 0, sizeof(unsigned int), h->stream));
    }
    if (groups) *groups = (int)c.enc_groups;
    if (bodies) *bodies = (int)c.enc_bodies;
    if (largest) *largest = (int)c.enc_maxsize;
    if (missed_pairs) *missed_pairs = (int)c.enc_missed;
    if (status) *status = (int)c.enc_status;
    return GENGA_OK;
}

int genga_encounter_work(genga_handle h, long long* rhs_total, int* rhs_max, int* rejected)
{
    if (!h || h->p.encounter_mode != 1) return GENGA_EINVAL;
    Counters c;
    std::memset(&c, 0, sizeof(c));
    if (h->N) {
        CU(cudaMemcpyAsync(&c, h->w.ctr, sizeof(c), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    if (rhs_total) *rhs_total = (long long)c.enc_rhs_sum;
    if (rhs_max) *rhs_max = (int)c.enc_rhs_max;
    if (rejected) *rejected = (int)c.enc_rejected;
    return GENGA_OK;
}

int genga_set_profiling(genga_handle h, int enable)
{
    if (!h) return GENGA_EINVAL;
    if (enable && !h->events_created) {
        for (int w = 0; w < Handle::NKT; ++w)
            for (int k = 0; k < Handle::EVPOOL; ++k) {
                CU(cudaEventCreate(&h->ev0[w][k]));
                CU(cudaEventCreate(&h->ev1[w][k]));
            }
        h->events_created = true;
    }
    if (!enable && h->prof) for (int w = 0; w < Handle::NKT; ++w) prof_flush(h, w);
    h->prof = enable & 15;
    return GENGA_OK;
}

int genga_kernel_time(genga_handle h, int which, double* ms_total, long long* launches, int reset)
{
    if (!h || which < 0 || which >= Handle::NKT) return GENGA_EINVAL;
    const int rc = prof_flush(h, which);
    if (rc != GENGA_OK) return rc;
    if (ms_total) *ms_total = h->ms_total[which];
    if (launches) *launches = h->ms_launches[which];
    if (reset) { h->ms_total[which] = 0.0; h->ms_launches[which] = 0; }
    return GENGA_OK;
}

long long genga_launch_count(genga_handle h) { return h ? h->launches : 0; }

int genga_synchronize(genga_handle h)
{
    if (!h) return GENGA_EINVAL;
    CU(cudaStreamSynchronize(h->stream));
    return GENGA_OK;
}

const char* genga_strerror(int code)
{
    switch (code) {
        case GENGA_OK:        return "ok";
        case GENGA_EINVAL:    return "invalid argument";
        case GENGA_ENOMEM:    return "workspace too small";
        case GENGA_ECAPACITY: return "encounter-pair list capacity exceeded";
        case GENGA_ECUDA:     return "CUDA error";
        case GENGA_ENOCONV:   return "Kepler solver did not converge";
        case GENGA_ELIMIT:    return "size beyond the fixed maximum of a no-allocation entry point (genga_static_last_error)";
        default:              return "unknown error";
    }
}

const char* genga_last_cuda_error(void) { return genga::g_cuda_err; }

const char* genga_version(void) { return "genga_b200 0.1 (sm_100a)"; }

int genga_set_tuning(genga_handle h, int key, int value)
{
    if (!h || key < 0 || key > 3) return GENGA_EINVAL;
    if (key >= 2) {                                    // grid of the all-pairs kernels in units of half a wave
        if (value < 0 || value > 64) return GENGA_EINVAL;
        h->tune[key] = value;
        return GENGA_OK;
    }
    const int n = key == 0 ? kick32_num_variants() : kick64_num_variants();
    if (value < 0 || value >= n) return GENGA_EINVAL;
    h->tune[key] = value;
    return GENGA_OK;
}

// Self-tuning in the sense of PAPER.md:55 ("tries configurations ... before the run"): time the
// force evaluation (prep + all-pairs + near field) of every variant on the current state and keep
// the fastest.  The state is not modified (only the acceleration / pair list of the last evaluation).
int genga_autotune(genga_handle h, int precision, int* chosen, double* ms_best)
{
    if (!h || (precision != GENGA_FP64 && precision != GENGA_FP32)) return GENGA_EINVAL;
    { const int rcf = flush_pending(h); if (rcf != GENGA_OK) return rcf; }
    const int key = precision == GENGA_FP32 ? 0 : 1;
    const int n = key == 0 ? kick32_num_variants() : kick64_num_variants();
    if (h->N == 0) { if (chosen) *chosen = h->tune[key]; if (ms_best) *ms_best = 0.0; return GENGA_OK; }
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
    const int prof = h->prof; h->prof = 0;
    int best = h->tune[key], rc = GENGA_OK;
    double best_ms = 1.0e300;
    for (int v = 0; v < n && rc == GENGA_OK; ++v) {
        h->tune[key] = v;
        if ((rc = force_eval(h, precision)) != GENGA_OK) break;             // warm-up (and first-use setup)
        double ms_min = 1.0e300;
        for (int rep = 0; rep < 3 && rc == GENGA_OK; ++rep) {
            cudaEventRecord(e0, h->stream);
            rc = force_eval(h, precision);
            cudaEventRecord(e1, h->stream);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = GENGA_ECUDA; break; }
            float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
            if (ms < ms_min) ms_min = ms;
        }
        if (rc == GENGA_OK && ms_min < best_ms) { best_ms = ms_min; best = v; }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    h->prof = prof;
    h->tune[key] = best;
    if (chosen) *chosen = best;
    if (ms_best) *ms_best = best_ms;
    return rc;
}

int genga_num_variants(int key)
{
    return key == 0 ? kick32_num_variants() : key == 1 ? kick64_num_variants() : 0;
}

const char* genga_variant_name(int key, int value)
{
    return key == 0 ? kick32_variant_name(value) : key == 1 ? kick64_variant_name(value) : "";
}

int genga_peak_probe(int which, int iters, void* stream, double* ops_per_s, double* ms)
{
    return run_peak_probe(which, iters, static_cast<cudaStream_t>(stream), ops_per_s, ms);
}

}  // extern "C"
