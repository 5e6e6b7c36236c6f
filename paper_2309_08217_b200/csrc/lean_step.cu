// lean_step.cu -- whole SEQUENCES of steps of a small system (N <= 2560) in one kernel with one grid-wide
// exchange per step and nothing else between the pair sums.
//
// The left end of the paper's Fig. 1 is bound by what happens BETWEEN the pair sums: kernel
// calls and, inside the one-kernel step of mega_step.cu, four grid-wide barriers and ~20 us of dependent
// phases at N = 1024.  Here a CTA OWNS a run of ~8 bodies (slots of the internal order) for the whole call:
// one thread per body keeps its velocity in registers and does the O(N) rows for it -- velocity update (a6),
// Sun-kick (a7, reading G3), Kepler drift (a8, FP64), critical radius (a1, Eq. 1) -- and the CTA's warps
// evaluate the COMPLETE pair sums of its bodies (a3 / a4, near pairs in FP64 with the changeover weight:
// a5) against the whole system, which every CTA holds in shared memory (80 bytes per body).  The
// accelerations therefore never leave the CTA; what the CTAs exchange per step is, after the drift, G partial
// sums of m v' and the drifted (x, |v|^2) of every body, 32 bytes per body: the closing Sun-kick needs
// P' = sum m v', pair sums and r_crit,ij need everybody's position.  The exchange (exchange_sums) is the one
// grid-wide barrier of the step; CTA 0 forms the total, so all CTAs hold bitwise the same P'.
// P = sum m v for the Sun-kick BEFORE the drift is summed once per call: a kick does not change it (DESIGN.md
// reading R17).  The closing velocity update of the sequence stays deferred (api.cu: sequence).
//
// FP32 policy P32 in this kernel: the frame is the CTA's (centre of the bounding box
// of ITS bodies; every j-position is rounded once per CTA and step relative to it), and the near bound is
// tested per PAIR in a separable form: r^2 <= max(c_i, c_j, Rf^2) takes the pair out of the FP32 (or
// refined-rsqrt FP64) sums, with c = (hq Amax)^2 >= (max(hq_i, hq_j) max(aq_i, aq_j))^2 for the mutual-Hill
// rule (Amax: the largest semi-major axis among the bodies within four times the mean; the others get
// c = inf) and c = (lambda r_crit)^2 for the max rule; Rf = max(largest rf of the system, frame guard of
// the CTA).  The bound parameters are FP32 UPPER bounds (rounded outwards with margins).  Such a pair gets
// its term in FP64 (near_pair): outside lambda^-1 of the bound the plain Newtonian term (it is certainly
// outside its changeover zone), else the exact term with r_crit,ij recomputed in FP64 from shared memory.
//
// -DLEAN_STAMPS (GENGA_NVCC_EXTRA) builds in %globaltimer stamps per phase and CTA and a printf of their
// mean and maximum over the CTAs at the end of a launch of 30 or more evaluations (a debugging build).
#include <cooperative_groups.h>
#ifdef LEAN_STAMPS
#include <cstdio>
#endif

#include "genga_internal.cuh"
#include "kepler.cuh"
#include "momentum.cuh"
#include "nearfield_body.cuh"

namespace genga {

namespace {

constexpr int LEAN_NT = 512;
constexpr int LEAN_NW = LEAN_NT / 32;
constexpr int LEAN_NMAX = 2560;                    // 80 bytes of shared memory per body
constexpr int LEAN_QCAP = 256;                     // near pairs a CTA queues per evaluation (more: evaluated on the spot)
constexpr int LEAN_SLOTW = 2048;                   // words of one array of exchange slots: 8 per CTA, at most 256 CTAs
static_assert(4 * LEAN_SLOTW == LEANX_WORDS, "two exchange arrays of slots and mailboxes");
constexpr int LEAN_NB = 8;                         // bodies a CTA owns, if there are SMs enough (measured: 4, 8, 16, 32)

struct LeanArgs {
    PrepArgs prep;
    nf::NfParams nfp;
    int lead, n_sds, pend;                         // [K(tau_first)] then n_sds x [S D S K]; pend: v += tau_prev a first
    double tau_prev, tau_first, tau_mid;
    double dt, mu;
    double* aout;                                  // accelerations of the last evaluation (not w.a: that one is still being read)
    int NI, JS, JL;                                // i-groups in all; warps per i-group (split of the j range), j-bodies per split
    int npart, nbmax;                              // doubles of the partial-sum scratch; most bodies a CTA owns
    unsigned long long seq0;                       // exchanges the handle has done before this launch (exchange_sums)
};

// shared memory of one CTA: the whole system
template <bool F32>
struct LeanSm {
    double *X, *Y, *Z, *GM;                        // [Nr] positions, G m
    double *M, *H, *V2;                            // [Nr] what the exact pair rule needs besides: m, cbrt(m / 3 M), |v|^2
    float4* R;                                     // [Nr] FP32 kernel: (x - o, G m) in the CTA's frame
    double* part;                                  // [npart] partial sums of the split j ranges / reduction scratch
    double* aloc;                                  // [3 nbmax] accelerations of the CTA's bodies
    float*  C;                                     // [Nr] separable near bound c_j
    float*  HQ;                                    // [Nr] its per-body factor, fixed for the call (hq_j; max rule: cbrt(m_j / 3 M) rounded up)
    int4*   queue;                                 // [LEAN_QCAP] near pairs of the evaluation: (si, sj, zone bound, -)
    int Nr;
};

template <bool F32>
__host__ __device__ inline size_t lean_smem_bytes(int N, int npart, int nbmax)
{
    const size_t Nr = (size_t)((N + 31) & ~31);
    return Nr * (F32 ? 80 : 64) + ((size_t)npart + 3 * (size_t)nbmax) * 8 + (size_t)LEAN_QCAP * 16;
}

template <bool F32>
__device__ __forceinline__ LeanSm<F32> lean_carve(unsigned char* raw, int N, int npart, int nbmax)
{
    const size_t Nr = (size_t)((N + 31) & ~31);
    LeanSm<F32> S;
    S.Nr = (int)Nr;
    S.queue = reinterpret_cast<int4*>(raw);
    S.X = reinterpret_cast<double*>(raw + (size_t)LEAN_QCAP * 16); S.Y = S.X + Nr; S.Z = S.Y + Nr; S.GM = S.Z + Nr;
    S.M = S.GM + Nr; S.H = S.M + Nr; S.V2 = S.H + Nr;
    double* q = S.V2 + Nr;
    if (F32) { S.R = reinterpret_cast<float4*>(q); q += 2 * Nr; } else S.R = nullptr;
    S.part = q; q += npart;
    S.aloc = q; q += 3 * nbmax;
    S.C = reinterpret_cast<float*>(q);
    S.HQ = S.C + Nr;
    return S;
}

// semi-major axis from vis-viva (readings G2b, G2c) exactly as prep_tile.cuh forms it
__device__ __forceinline__ double semi_axis(double px, double py, double pz, double v2, double mu)
{
    const double r = sqrt(px * px + py * py + pz * pz);
    double sa = 1.0 / (2.0 / r - v2 / mu);
    if (!(sa > 0.0) || !isfinite(sa)) sa = r;
    return sa;
}

struct Vec3 { double x, y, z; };

// |v|^2 of a body at the start of the call: the stored velocity with the owed update
__device__ __forceinline__ double speed2_start(const LeanArgs& L, const Workspace& w, int body)
{
    double v0 = w.v[3 * body], v1 = w.v[3 * body + 1], v2 = w.v[3 * body + 2];
    if (L.pend) { v0 = fma(L.tau_prev, w.a[3 * body], v0); v1 = fma(L.tau_prev, w.a[3 * body + 1], v1); v2 = fma(L.tau_prev, w.a[3 * body + 2], v2); }
    return v0 * v0 + v1 * v1 + v2 * v2;
}

// The exact FP64 term of body (slot) sj on body si for a pair that may lie inside its changeover zone, as
// nearfield_body.cuh: chunk_on_body phase B computes it (plain sqrt / divide / cbrt, r_crit,ij by the pair rule O3,
// weight O4), and the encounter list if `list`.  Everything it needs is in shared memory.
__device__ __noinline__ Vec3 exact_pair(const double* X, int Nr, const LeanArgs& L, const Workspace& w, int si, int sj, bool list)
{
    const double *Y = X + Nr, *Z = Y + Nr, *GM = Z + Nr, *M = GM + Nr, *H = M + Nr, *V2 = H + Nr;
    const nf::NfParams& P = L.nfp;
    Vec3 f = {0.0, 0.0, 0.0};
    const double sai = semi_axis(X[si], Y[si], Z[si], V2[si], L.mu), saj = semi_axis(X[sj], Y[sj], Z[sj], V2[sj], L.mu);
    const double vki = sqrt(L.mu / sai), vkj = sqrt(L.mu / saj);
    const double rci = fmax(P.n1 * (sai * H[si]), P.n2dt * vki);
    const double rcj = fmax(P.n1 * (saj * H[sj]), P.n2dt * vkj);
    const double dx = X[sj] - X[si], dy = Y[sj] - Y[si], dz = Z[sj] - Z[si];
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const double r  = sqrt(r2);
    const double rc = nf::pair_rcrit(P, M[si], M[sj], rci, rcj, sai, saj, vki, vkj);
    if (list && (si < sj) && (r < P.list_scale * rc)) {                       // coincident bodies (r = 0) are an encounter
        const unsigned int idx = atomicAdd(&w.ctr->pair_count, 1u);
        const int bi = w.order[si], bj = w.order[sj];
        if (idx < P.pair_cap) w.pairs[idx] = make_int2(min(bi, bj), max(bi, bj));
    }
    if (r > 0.0) {
        const double W = nf::changeover(r, rc, P.weight_mode);
        if (W != 0.0) {
            const double s = GM[sj] * W / (r2 * r);
            f.x = s * dx; f.y = s * dy; f.z = s * dz;
        }
    }
#ifdef LEAN_STAMPS
    atomicAdd(&w.ctr->cand_count, 1u);
#endif
    return f;
}

// A pair inside its near bound: outside lambda^-1 of the bound it is certainly outside its changeover zone (the bound is
// lambda times an upper bound of r_crit,ij), W = 1 and it cannot be an encounter: the plain FP64 term.  Otherwise exact_pair.
// zc: max(c_i, c_j, Rf_orbit^2) / lambda^2 of the pair (the frame guard is not part of it).
template <bool F32>
__device__ __forceinline__ void near_pair(const LeanSm<F32>& S, const LeanArgs& L, const Workspace& w, int si, int sj, float zc, bool list,
                                          double& fx, double& fy, double& fz)
{
    const double dx = S.X[sj] - S.X[si], dy = S.Y[sj] - S.Y[si], dz = S.Z[sj] - S.Z[si];
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    if (r2 > (double)zc) {
        const double s = S.GM[sj] / (r2 * sqrt(r2));
        fx = fma(s, dx, fx); fy = fma(s, dy, fy); fz = fma(s, dz, fz);
#ifdef LEAN_STAMPS
        atomicAdd(&w.ctr->overflow, 1u);
#endif
    } else {
        const Vec3 f = exact_pair(S.X, S.Nr, L, w, si, sj, list);
        fx += f.x; fy += f.y; fz += f.z;
    }
}

__host__ __device__ constexpr int lean_ib(bool f32) { return f32 ? 4 : 2; }              // bodies per warp pass

// The O(N^2) row for the i-groups [g0, g1) of this CTA: one warp per (i-group, j-range), complete sums over j after
// the ranges' partials are added in a fixed order -> aloc[3 (s - s_lo) + c].  A pass of a warp is free of calls and
// branches: IB bodies against 32 j-bodies; FP32 kernel: FP32 terms summed in FP32 per lane (at most N / 32 terms),
// lanes and ranges combined in FP64; FP64 kernel: the refined-rsqrt term of nearfield_body.cuh.  A pair inside its near
// bound contributes nothing there: bit `it` of a lane's mask records it, and after a block of 32 passes the lane looks at
// its flagged pairs in FP64: outside lambda^-1 of its bound a pair is certainly outside its changeover zone and gets
// the plain FP64 term at once; the others are queued (si, sj, zone bound) for the whole CTA, which evaluates them
// (near_pair -> exact_pair), one thread per pair, and adds the terms to aloc (atomically: the order of these few
// additions is not fixed).  A pair that finds the queue full is evaluated on the spot.  rfg2: Rf^2 of this CTA (see the head of the file); rfo2: without the frame
// guard; ilam2: lambda^-2 rounded up; list: append the encounter pairs to the list (the last evaluation of the call).
template <bool F32>
__device__ __forceinline__ void lean_kick(const LeanSm<F32>& S, const LeanArgs& L, const Workspace& w, int N, int g0, int g1,
                                          float rfg2, float rfo2, float ilam2, bool list, int* qn)
{
    constexpr int IB = lean_ib(F32);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int nitem = (g1 - g0) * L.JS;
    const int s_lo = g0 * IB;
    if (threadIdx.x == 0) *qn = 0;
    __syncthreads();
    for (int item = wid; item < nitem; item += LEAN_NW) {
        const int ig = item / L.JS, js = item - ig * L.JS;
        const int si0 = (g0 + ig) * IB;
        const int j0 = js * L.JL, j1 = min(N, j0 + L.JL);
        double ex[IB], ey[IB], ez[IB];
        int sib[IB];
        float cn[IB], ci[IB];
#pragma unroll
        for (int b = 0; b < IB; ++b) {
            ex[b] = ey[b] = ez[b] = 0.0;
            sib[b] = (si0 + b < N) ? si0 + b : -1;
            cn[b] = sib[b] >= 0 ? S.C[sib[b]] : 0.f;
            ci[b] = fmaxf(cn[b], rfg2);
        }
        float xi[IB], yi[IB], zi[IB], ax[IB], ay[IB], az[IB];                 // FP32 kernel
        double xd[IB], yd[IB], zd[IB];                                        // FP64 kernel
#pragma unroll
        for (int b = 0; b < IB; ++b) {
            ax[b] = ay[b] = az[b] = 0.f;
            xi[b] = yi[b] = zi[b] = 0.f; xd[b] = yd[b] = zd[b] = 0.0;
            if (sib[b] >= 0) {
                if constexpr (F32) { const float4 q = S.R[sib[b]]; xi[b] = q.x; yi[b] = q.y; zi[b] = q.z; }
                else               { xd[b] = S.X[sib[b]]; yd[b] = S.Y[sib[b]]; zd[b] = S.Z[sib[b]]; }
            }
        }
        for (int jbase = j0; jbase < j1; jbase += 1024) {
            const int jb = jbase + lane;
            unsigned int mask[IB];
#pragma unroll
            for (int b = 0; b < IB; ++b) mask[b] = 0u;
            const int nit = jb < j1 ? min(32, (j1 - jb + 31) >> 5) : 0;
            if constexpr (F32) {
#pragma unroll 2
                for (int it = 0; it < nit; ++it) {
                    const int j = jb + 32 * it;
                    const float4 q = S.R[j];
                    const float cj = S.C[j];
                    const unsigned int bit = 1u << it;
#pragma unroll
                    for (int b = 0; b < IB; ++b) {
                        const float dx = q.x - xi[b], dy = q.y - yi[b], dz = q.z - zi[b];
                        const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                        const bool near = !(r2 > fmaxf(ci[b], cj));
                        const float y = rsqrtf(r2);
                        const float s = near ? 0.f : (q.w * y) * (y * y);
                        ax[b] = fmaf(s, dx, ax[b]); ay[b] = fmaf(s, dy, ay[b]); az[b] = fmaf(s, dz, az[b]);
                        if (near) mask[b] |= bit;
                    }
                }
            } else {
#pragma unroll 2
                for (int it = 0; it < nit; ++it) {
                    const int j = jb + 32 * it;
                    const double xj = S.X[j], yj = S.Y[j], zj = S.Z[j], gj = S.GM[j];
                    const float cj = S.C[j];
                    const unsigned int bit = 1u << it;
#pragma unroll
                    for (int b = 0; b < IB; ++b) {
                        const double dx = xj - xd[b], dy = yj - yd[b], dz = zj - zd[b];
                        const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                        const bool near = !(__double2float_rd(r2) > fmaxf(ci[b], cj));
                        const double y0 = nf::rsq64h(r2);
                        const double tt = y0 * y0;
                        const double e  = fma(-r2, tt, 1.0);
                        const double cc = fma(1.875, e, 1.5);
                        const double g  = (gj * y0) * tt;
                        const double s  = near ? 0.0 : fma(g * e, cc, g);
                        ex[b] = fma(s, dx, ex[b]); ey[b] = fma(s, dy, ey[b]); ez[b] = fma(s, dz, ez[b]);
                        if (near) mask[b] |= bit;
                    }
                }
            }
#pragma unroll
            for (int b = 0; b < IB; ++b) {
                if (!__any_sync(0xffffffffu, mask[b] != 0u)) continue;
                unsigned int m = sib[b] >= 0 ? mask[b] : 0u;
                while (m) {
                    const int j = jb + 32 * (__ffs(m) - 1);
                    m &= m - 1u;
                    if (j == sib[b]) continue;
                    const float zc = fmaxf(fmaxf(cn[b], S.C[j]), rfo2) * ilam2;
                    const double dx = S.X[j] - S.X[sib[b]], dy = S.Y[j] - S.Y[sib[b]], dz = S.Z[j] - S.Z[sib[b]];
                    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                    if (r2 > (double)zc) {                                   // certainly outside its zone: the plain FP64 term, here and now
                        const double s = S.GM[j] / (r2 * sqrt(r2));
                        ex[b] = fma(s, dx, ex[b]); ey[b] = fma(s, dy, ey[b]); ez[b] = fma(s, dz, ez[b]);
                        continue;
                    }
                    const int k = atomicAdd(qn, 1);
                    if (k < LEAN_QCAP) S.queue[k] = make_int4(sib[b], j, __float_as_int(zc), 0);
                    else near_pair<F32>(S, L, w, sib[b], j, zc, list, ex[b], ey[b], ez[b]);
                }
            }
        }
#pragma unroll
        for (int b = 0; b < IB; ++b) {
            if constexpr (F32) { ex[b] += (double)ax[b]; ey[b] += (double)ay[b]; ez[b] += (double)az[b]; }
            const double fx = nf::warp_sum(ex[b]), fy = nf::warp_sum(ey[b]), fz = nf::warp_sum(ez[b]);
            if (lane == 0) {
                double* p = S.part + (size_t)(item * IB + b) * 3;
                p[0] = fx; p[1] = fy; p[2] = fz;
            }
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < (g1 - g0) * IB * 3; t += LEAN_NT) {
        const int ig = t / (IB * 3), r = t - ig * (IB * 3);
        double s = 0.0;
        for (int js = 0; js < L.JS; ++js) s += S.part[(size_t)(ig * L.JS + js) * IB * 3 + r];
        S.aloc[t] = s;                                                        // t = 3 (s - s_lo) + c
    }
    const int nq = min(*qn, LEAN_QCAP);
    __syncthreads();
    if (nq > 0) {
        for (int k = threadIdx.x; k < nq; k += LEAN_NT) {
            const int4 en = S.queue[k];
            double fx = 0.0, fy = 0.0, fz = 0.0;
            near_pair<F32>(S, L, w, en.x, en.y, __int_as_float(en.z), list, fx, fy, fz);
            double* a = S.aloc + 3 * (en.x - s_lo);
            atomicAdd(a, fx); atomicAdd(a + 1, fy); atomicAdd(a + 2, fz);
        }
        __syncthreads();
    }
}

// Grid-wide sum of one (p0, p1, p2, mt) per CTA that is a barrier at the same time.  A CTA publishes its four sums as
// four 16-byte words (value, seq) in its slot; CTA 0 (warp 0) polls the G slots until each word carries seq, adds the
// values in a fixed order and publishes the four totals the same way in slot G; every CTA polls only that slot, so all
// CTAs get the same bits.  seq grows with every exchange of the handle's life: a slot never has to be cleared.  A word
// is written and read with one aligned 16-byte access, which the hardware does not tear (NCCL's LL protocols lean on
// the same property), so the values need no flag of their own and no fence.  fence = true also orders the OTHER global
// writes of every CTA (the drifted positions) before the reads that follow the exchange in any CTA: release before the
// publishing, acquire after the polling, passed on through CTA 0.  Needs all CTAs co-resident (cooperative launch).
__device__ __forceinline__ void lean_fence() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ void ll_store(unsigned long long* q, double v, unsigned long long seq)
{
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" :: "l"(q), "l"((unsigned long long)__double_as_longlong(v)), "l"(seq) : "memory");
}
__device__ __forceinline__ bool ll_load(const unsigned long long* q, unsigned long long seq, double& val)
{
    unsigned long long v, f;
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(v), "=l"(f) : "l"(q) : "memory");
    val = __longlong_as_double((long long)v);
    return f >= seq;
}
__device__ __forceinline__ void exchange_sums(double p0, double p1, double p2, double mt, int nw, double* scratch,
                                              unsigned long long* slots, int G, unsigned long long seq, bool fence, double* out4)
{
    warp_sum4(p0, p1, p2, mt);
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0 && wid < nw) { scratch[4 * wid] = p0; scratch[4 * wid + 1] = p1; scratch[4 * wid + 2] = p2; scratch[4 * wid + 3] = mt; }
    __syncthreads();
    if (wid == 0 && lane < 4) {                                           // lane c: sum c of the owners' warps, published
        double v = 0.0;
        for (int k = 0; k < nw; ++k) v += scratch[4 * k + lane];
        if (fence) lean_fence();
        ll_store(slots + 8 * (size_t)blockIdx.x + 2 * lane, v, seq);
    }
    if (blockIdx.x == 0) {
        // CTA 0: thread t waits for the words t and t + LEAN_NT of the G slots (word = 4 slot + component: G <= 256), then
        // the sum over the slots per component: lanes with equal (lane & 3) inside a warp, the warps through shared memory
        double v0 = 0.0, v1 = 0.0;
        const int w0 = threadIdx.x, w1 = threadIdx.x + LEAN_NT;
        bool ok0 = w0 >= 4 * G, ok1 = w1 >= 4 * G;
        while (!(ok0 && ok1)) {
            if (!ok0) ok0 = ll_load(slots + 2 * (size_t)w0, seq, v0);
            if (!ok1) ok1 = ll_load(slots + 2 * (size_t)w1, seq, v1);
        }
        if (fence) lean_fence();                                       // acquire: what the CTAs wrote before they published
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) { v0 += __shfl_xor_sync(0xffffffffu, v0, o); v1 += __shfl_xor_sync(0xffffffffu, v1, o); }
        __syncthreads();                                                  // the owners' partials in scratch have been read
        if (lane < 4) scratch[4 * wid + lane] = v0 + v1;
        __syncthreads();
        if (wid == 0) {
            // warp 0: the LEAN_NW warps' sums in a fixed tree, then the totals to the mailboxes of the CTAs (word 4 b + c of
            // the second half of the array: every CTA polls its own four words only)
            static_assert(LEAN_NW == 16, "two values per lane");
            double tot = scratch[lane] + scratch[lane + 32];
#pragma unroll
            for (int o = 4; o < 32; o <<= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
            if (fence) lean_fence();                                   // ... is passed on with the totals (release)
            unsigned long long* box = slots + LEAN_SLOTW;
            for (int k = lane; k < 4 * G; k += 32) ll_store(box + 2 * (size_t)k, tot, seq);   // k & 3 == lane & 3: this lane's component
        }
    }
    if (wid == 0) {
        if (lane < 4) { double v; while (!ll_load(slots + LEAN_SLOTW + 8 * (size_t)blockIdx.x + 2 * lane, seq, v)) { } out4[lane] = v; }
        if (fence) lean_fence();
    }
    __syncthreads();
}

// FP32 UPPER bounds of the semi-major axis and of v_K^2 = G M / a from (x, |v|^2): every rounding error of the FP32
// evaluation of d = 2/r - v^2/mu is below 5e-7 (2/r + v^2/mu); a body whose d may have either sign gets a = 3e38
// (all its pairs take the exact term), a certainly unbound one a = r (the fallback of semi_axis).
__device__ __forceinline__ void bound_orbit(float x, float y, float z, float v2, float mu, float imu, float& aq, float& vk2)
{
    const float r2 = fmaf(z, z, fmaf(y, y, x * x));
    const float ri = rsqrtf(r2);
    const float a = 2.0f * ri, b = v2 * imu;
    const float d = a - b, del = 2.0e-6f * (a + b);
    const float dlo = d - del, dhi = d + del;
    if (dlo > 0.f)      aq = __fdividef(1.000002f, dlo) * 1.000002f;
    else if (dhi < 0.f) aq = (r2 * ri) * 1.000004f;
    else                aq = 3.0e38f;
    vk2 = mu * fmaxf(dhi, ri * 1.000002f) * 1.000002f;
    if (!(aq >= 0.f)) aq = 3.0e38f;
    if (!(vk2 >= 0.f)) vk2 = 3.0e38f;
}

// max or sum over the CTA of one float per thread, through buf[LEAN_NW]; every thread returns the result
template <bool MAX>
__device__ __forceinline__ float block_reduce_f(float v, float* buf)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float u = __shfl_xor_sync(0xffffffffu, v, o);
        v = MAX ? fmaxf(v, u) : v + u;
    }
    if ((threadIdx.x & 31) == 0) buf[threadIdx.x >> 5] = v;
    __syncthreads();
    float r = buf[0];
#pragma unroll
    for (int k = 1; k < LEAN_NW; ++k) r = MAX ? fmaxf(r, buf[k]) : r + buf[k];
    return r;
}

// Tau of the velocity update that precedes evaluation e (e >= 1): the kick evaluation e - 1 belongs to.
__device__ __forceinline__ double tau_before(const LeanArgs& L, int e)
{
    return (L.lead && e == 1) ? L.tau_first : L.tau_mid;
}

template <bool F32>
__global__ void __launch_bounds__(LEAN_NT, 1)
lean_kernel(const __grid_constant__ LeanArgs L, const __grid_constant__ Workspace w)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    __shared__ double sP[4];
    __shared__ double sO[4];
    __shared__ float sF[2];
    __shared__ int sQn;
    __shared__ float sR1[LEAN_NW], sR2[LEAN_NW], sR3[LEAN_NW], sR4[LEAN_NW];
    const LeanSm<F32> S = lean_carve<F32>(smraw, L.prep.N, L.npart, L.nbmax);
    const PrepArgs& A = L.prep;
    const int N = A.N, t = threadIdx.x, lane = t & 31, wid = t >> 5;
    const int G = (int)gridDim.x, cta = (int)blockIdx.x;
    const int E = L.lead + L.n_sds;
    constexpr int IB = lean_ib(F32);
    const int g0 = (int)(((long long)L.NI * cta) / G), g1 = (int)(((long long)L.NI * (cta + 1)) / G);
    const int s_lo = g0 * IB, s_hi = min(N, g1 * IB);            // this CTA's bodies
    const int nb = s_hi - s_lo, nwo = (nb + 31) >> 5;             // ... and the warps of their owner threads
    const bool hill = A.pair_rule == GENGA_PAIR_MUTUAL_HILL;
    const double lam = (double)A.lambda * (1.0 + 1.0e-6);
    const float muf = __double2float_ru(L.mu), imuf = __double2float_ru(1.0 / L.mu);
    const float ilam2 = __double2float_ru(1.00001 / ((double)A.lambda * (double)A.lambda));
    // exchange arrays of P and of P': LEAN_SLOTW words for the CTAs' sums (8 per CTA), then as many for the mailboxes
    unsigned long long* pg1 = w.leanx;
    unsigned long long* pg2 = pg1 + 2 * LEAN_SLOTW;
    unsigned long long seq = L.seq0;
    // the drifted (x, |v|^2) of every slot, in two buffers that alternate from step to step: with one exchange per step a fast
    // CTA may publish step e + 1 while a slow one is still loading step e; it cannot get to step e + 2 before that one has
    // published step e + 1, i.e. is done loading
    double4* const xgb[2] = {w.pk64, w.aux};

    // per-thread part of the near bounds of an evaluation (see below): bound_orbit of every slot this thread loads
    const float n2dtf = __double2float_ru(lam * A.n2 * A.dt_rcrit);
    const float ln1f = __double2float_ru(lam * A.n1);
    float asum = 0.f, acnt = 0.f, vkmax = 0.f, amax_t = 0.f;
    float cap = -1.f;                                         // mutual-Hill rule: 4 x the mean semi-major axis, fixed at the first evaluation of the call
    auto note_orbit = [&](int s, double px, double py, double pz, double v2) {
        float aq, vk2;
        bound_orbit((float)px, (float)py, (float)pz, __double2float_ru(v2), muf, imuf, aq, vk2);
        if (hill) {
            S.C[s] = aq;                                          // turned into c_s once Amax is known
            if (cap < 0.f) { if (aq < 1.0e30f) { asum += aq; acnt += 1.f; } }
            else if (aq <= cap) amax_t = fmaxf(amax_t, aq);
            vkmax = fmaxf(vkmax, vk2);
        } else {
            // max rule: c = (lambda r_crit)^2 from the upper bounds (HQ: cbrt(m / 3 M) rounded up)
            const float rc = fmaxf(ln1f * (aq * S.HQ[s]), n2dtf * (sqrtf(vk2) * 1.000001f)) * 1.000002f;
            float c = rc * rc * 1.000001f;
            if (!(c >= 0.f)) c = 3.0e38f;
            S.C[s] = c;
        }
    };

    // ---- the system at the start of the call -------------------------------------------------------------
    for (int s = t; s < N; s += LEAN_NT) {
        const int i = w.order[s];
        const double px = w.x[3 * i], py = w.x[3 * i + 1], pz = w.x[3 * i + 2];
        S.X[s] = px; S.Y[s] = py; S.Z[s] = pz;
        const double mi = w.m[i], h = w.hcbrt[i];
        S.GM[s] = A.G * mi;
        if (F32) S.R[s] = make_float4(0.f, 0.f, 0.f, (float)(A.G * mi));
        float hq = hill ? __fmul_ru(__double2float_ru(lam * A.n1 * 1.2599210498948732 * h), 1.000001f) : __double2float_ru(h);
        if (!(hq >= 0.f)) hq = 3.0e38f;
        S.HQ[s] = hq;
        S.M[s] = mi; S.H[s] = h;
        if (L.lead) { const double v2 = speed2_start(L, w, i); S.V2[s] = v2; note_orbit(s, px, py, pz, v2); }   // the first evaluation is at these positions
    }
    const bool own = t < nb;
    const int so = s_lo + t;                                      // the slot thread t owns
    int bo = -1;
    double mo = 0.0, vx = 0.0, vy = 0.0, vz = 0.0;
    if (own) { bo = w.order[so]; mo = w.m[bo]; vx = w.v[3 * bo]; vy = w.v[3 * bo + 1]; vz = w.v[3 * bo + 2]; }
    if (cta == 0 && t == 0) { w.ctr->cand_count = 0u; w.ctr->overflow = 0u; }
    __syncthreads();

#ifdef LEAN_STAMPS
    unsigned long long st_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, st_t = 0;
#define LEAN_STAMP(k) do { if (t == 0) { unsigned long long n_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(n_)); st_acc[k] += n_ - st_t; st_t = n_; } } while (0)
    if (t == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(st_t));
#else
#define LEAN_STAMP(k)
#endif
    for (int e = 0; e < E; ++e) {
        const bool drift = e >= L.lead;
        const bool last = e == E - 1;
        // ---- row a6: close the previous kick (own bodies) -----------------------------------------------
        if (own && (e > 0 || L.pend)) {
            if (e > 0) {
                const double tau = tau_before(L, e);
                vx = fma(tau, S.aloc[3 * t], vx); vy = fma(tau, S.aloc[3 * t + 1], vy); vz = fma(tau, S.aloc[3 * t + 2], vz);
            } else {
                vx = fma(L.tau_prev, w.a[3 * bo], vx); vy = fma(L.tau_prev, w.a[3 * bo + 1], vy); vz = fma(L.tau_prev, w.a[3 * bo + 2], vz);
            }
        }
        if (drift) {
            // ---- P = sum m v; rows a7, a8: S(dt/2) D(dt); P' = sum m v' -----------------------------------
            const double sc = 0.5 * L.dt / A.M_star;
            // P = sum m v is summed at the first drift of the call only: a kick does not change it (the pair forces are equal
            // and opposite: sum m a = 0 up to the rounding of the pair terms), so later steps go on with the P' = sum m v' that
            // the previous step summed after its drift (reading R17)
            if (e == L.lead)
                exchange_sums(own ? mo * vx : 0.0, own ? mo * vy : 0.0, own ? mo * vz : 0.0, own ? mo : 0.0, nwo, S.part, pg1, G, ++seq, false, sP);
            LEAN_STAMP(0);
            if (last && cta == 0 && t < 4) w.mom[MOM_SLOT_A + t] = sP[t];
            double p0 = 0, p1 = 0, p2 = 0, mt = 0;
            if (own) {
                double x0 = S.X[so] + sc * sP[0], y0 = S.Y[so] + sc * sP[1], z0 = S.Z[so] + sc * sP[2];
                if (L.dt != 0.0) { if (!kepler_drift(L.mu, L.dt, x0, y0, z0, vx, vy, vz)) atomicAdd(&w.ctr->noconv, 1u); }
                double2* g2 = reinterpret_cast<double2*>(&xgb[e & 1][so]);
                __stcg(g2, make_double2(x0, y0)); __stcg(g2 + 1, make_double2(z0, vx * vx + vy * vy + vz * vz));
                p0 = mo * vx; p1 = mo * vy; p2 = mo * vz; mt = mo;
            }
            LEAN_STAMP(1);
            exchange_sums(p0, p1, p2, mt, nwo, S.part, pg2, G, ++seq, true, sP);
            LEAN_STAMP(2);
            if (last && cta == 0 && t < 4) w.mom[MOM_SLOT_B + t] = sP[t];
            // closing S(dt/2): everybody's position, shifted as its owner shifts it
            const double s0 = sc * sP[0], s1 = sc * sP[1], s2 = sc * sP[2];
            asum = acnt = vkmax = amax_t = 0.f;
            for (int s = t; s < N; s += LEAN_NT) {
                const double2* g2 = reinterpret_cast<const double2*>(&xgb[e & 1][s]);
                const double2 qa = __ldcg(g2), qb = __ldcg(g2 + 1);
                const double px = qa.x + s0, py = qa.y + s1, pz = qb.x + s2;
                S.X[s] = px; S.Y[s] = py; S.Z[s] = pz; S.V2[s] = qb.y;
                note_orbit(s, px, py, pz, qb.y);
            }
            __syncthreads();
        }
        // ---- rows a1, a2: the state the call leaves behind (last evaluation); near bounds of everybody -----
        if (last && e == 0 && L.lead) exchange_sums(0.0, 0.0, 0.0, 0.0, nwo, S.part, pg1, G, ++seq, true, sO);   // everybody has read the old state
        if (last && own) {
            const double px = S.X[so], py = S.Y[so], pz = S.Z[so];
            const double sa = semi_axis(px, py, pz, vx * vx + vy * vy + vz * vz, L.mu);
            const double vk = sqrt(L.mu / sa);
            w.x[3 * bo] = px; w.x[3 * bo + 1] = py; w.x[3 * bo + 2] = pz;
            w.v[3 * bo] = vx; w.v[3 * bo + 1] = vy; w.v[3 * bo + 2] = vz;
            w.rcrit[bo] = fmax(A.n1 * (sa * w.hcbrt[bo]), A.n2 * A.dt_rcrit * vk); w.semi[bo] = sa; w.vkep[bo] = vk;
        }
        // near bounds of everybody (bound_orbit was taken when the positions were loaded): Amax, then c_s
        // (Any cap gives a valid bound: a body beyond it gets c = inf, i.e. all its pairs in FP64.  So the cap of the call's
        // first evaluation serves the later ones, whose loading loop then collects Amax on the way: one reduction per step.)
        float rfo = 0.f, amax = 0.f;
        if (hill) {
            if (cap < 0.f) {
                asum = block_reduce_f<false>(asum, sR1);
                acnt = block_reduce_f<false>(acnt, sR2);
                cap = 4.0f * asum / fmaxf(acnt, 1.f);
                if (!(cap >= 0.f)) cap = 0.f;                 // (NaN state: everything in FP64)
                for (int s = t; s < N; s += LEAN_NT) { const float aq = S.C[s]; if (aq <= cap) amax_t = fmaxf(amax_t, aq); }
            }
            amax = block_reduce_f<true>(amax_t, sR3);
            if (A.n2 * A.dt_rcrit != 0.0) rfo = n2dtf * (sqrtf(block_reduce_f<true>(vkmax, sR4)) * 1.000001f) * 1.000002f;
        }
        auto hill_c = [&](int s) {                            // c_s from a_s (left in C by the loading loop) and Amax
            const float tq = S.HQ[s] * amax;
            float c = (S.C[s] <= cap) ? tq * tq * 1.000001f : 3.0e38f;
            if (!(c >= 0.f)) c = 3.0e38f;
            return c;
        };
        if (hill && !F32)
            for (int s = t; s < N; s += LEAN_NT) S.C[s] = hill_c(s);
        // warp 0: origin of the CTA's frame (centre of the bounding box of its bodies) and their radius about it
        if (wid == 0) {
            float lo0 = 3.0e38f, lo1 = 3.0e38f, lo2 = 3.0e38f, hi0 = -3.0e38f, hi1 = -3.0e38f, hi2 = -3.0e38f;
            for (int s = s_lo + lane; s < s_hi; s += 32) {
                const float fx = (float)S.X[s], fy = (float)S.Y[s], fz = (float)S.Z[s];
                lo0 = fminf(lo0, fx); hi0 = fmaxf(hi0, fx); lo1 = fminf(lo1, fy); hi1 = fmaxf(hi1, fy);
                lo2 = fminf(lo2, fz); hi2 = fmaxf(hi2, fz);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                lo0 = fminf(lo0, __shfl_xor_sync(0xffffffffu, lo0, o)); hi0 = fmaxf(hi0, __shfl_xor_sync(0xffffffffu, hi0, o));
                lo1 = fminf(lo1, __shfl_xor_sync(0xffffffffu, lo1, o)); hi1 = fmaxf(hi1, __shfl_xor_sync(0xffffffffu, hi1, o));
                lo2 = fminf(lo2, __shfl_xor_sync(0xffffffffu, lo2, o)); hi2 = fmaxf(hi2, __shfl_xor_sync(0xffffffffu, hi2, o));
            }
            const bool any = lo0 <= hi0 && lo1 <= hi1 && lo2 <= hi2;     // false: no body (or a NaN state)
            const double ox = any ? (double)(0.5f * lo0 + 0.5f * hi0) : 0.0, oy = any ? (double)(0.5f * lo1 + 0.5f * hi1) : 0.0,
                         oz = any ? (double)(0.5f * lo2 + 0.5f * hi2) : 0.0;
            float rad = 0.f;
            for (int s = s_lo + lane; s < s_hi; s += 32) {
                const double qx = S.X[s] - ox, qy = S.Y[s] - oy, qz = S.Z[s] - oz;
                float r1 = __double2float_ru(sqrt(qx * qx + qy * qy + qz * qz) * (1.0 + 1.0e-9));
                if (!(r1 >= 0.f)) r1 = 3.0e38f;
                rad = fmaxf(rad, r1);
            }
            rad = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(rad)));
            if (lane == 0) {
                // frame guard: pairs closer than floor * 2 R go to FP64 (relative rounding error of the FP32 separation
                // <= 2^-24 (1 + 2 R / r)); never below 1e-12 length units, so that the FP32 term cannot overflow
                const float guard = F32 ? __fmul_ru(__fmul_ru(2.0f * A.floor_rel, rad), 1.000001f) : 0.f;
                const float rr = fmaxf(rfo, guard);
                float c = fmaxf(__fmul_ru(__fmul_ru(rr, rr), 1.000001f), 1.0e-24f);
                if (!(c >= 0.f)) c = 3.0e38f;
                sF[0] = c;
                float co = __fmul_ru(__fmul_ru(rfo, rfo), 1.000001f);
                if (!(co >= 0.f)) co = 3.0e38f;
                sF[1] = co;
                sO[0] = ox; sO[1] = oy; sO[2] = oz;
            }
        }
        __syncthreads();
        if (F32) {
            const double ox = sO[0], oy = sO[1], oz = sO[2];
            for (int s = t; s < N; s += LEAN_NT) {
                if (hill) S.C[s] = hill_c(s);
                S.R[s] = make_float4((float)(S.X[s] - ox), (float)(S.Y[s] - oy), (float)(S.Z[s] - oz), S.R[s].w);
            }
            __syncthreads();
        }
        LEAN_STAMP(3);
        // ---- rows a3 / a4 / a5: the complete sums of this CTA's bodies ----------------------------------
        lean_kick<F32>(S, L, w, N, g0, g1, sF[0], sF[1], ilam2, last, &sQn);
        LEAN_STAMP(4);
        if (last && own) { L.aout[3 * bo] = S.aloc[3 * t]; L.aout[3 * bo + 1] = S.aloc[3 * t + 1]; L.aout[3 * bo + 2] = S.aloc[3 * t + 2]; }
    }
#ifdef LEAN_STAMPS
    if (E >= 30) {
        unsigned long long* dbg = reinterpret_cast<unsigned long long*>(w.vtmp);
        if (t == 0) for (int k = 0; k < 5; ++k) __stcg(&dbg[8 * cta + k], st_acc[k]);
        exchange_sums(0.0, 0.0, 0.0, 0.0, nwo, S.part, pg1, G, ++seq, true, sO);
        if (t == 0 && cta == 0) {
            double mx[5] = {0, 0, 0, 0, 0}, mean[5] = {0, 0, 0, 0, 0};
            for (int b = 0; b < G; ++b) for (int k = 0; k < 5; ++k) { const double v = (double)__ldcg(&dbg[8 * b + k]) / E; mx[k] = fmax(mx[k], v); mean[k] += v / G; }
            printf("lean N=%d E=%d G=%d ns/eval mean|max over CTAs: P+bar1 %.0f|%.0f drift %.0f|%.0f bar2 %.0f|%.0f load+prep %.0f|%.0f kick %.0f|%.0f; zone pairs %.1f, plain %.1f\n",
                   N, E, G, mean[0], mx[0], mean[1], mx[1], mean[2], mx[2], mean[3], mx[3], mean[4], mx[4], (double)w.ctr->cand_count / E, (double)w.ctr->overflow / E);
        }
    }
#endif
}

struct LeanPlan { int G, NI, JS, JL, npart, nbmax; size_t smem; const void* fn; };

// How the bodies are shared out over at most `blocks` CTAs: NI i-groups in contiguous runs of about LEAN_NB bodies, and,
// while a CTA has fewer i-groups than warps, JS warps per i-group with a range of JL j-bodies each.
LeanPlan lean_plan(int N, int precision, int blocks)
{
    LeanPlan p;
    const bool f32 = precision == GENGA_FP32;
    const int IB = lean_ib(f32);
    p.NI = (N + IB - 1) / IB;
    p.G = (N + LEAN_NB - 1) / LEAN_NB;
    if (p.G > blocks) p.G = blocks;
    if (p.G > p.NI) p.G = p.NI;
    if (p.G < 1) p.G = 1;
    const int ngmax = (p.NI + p.G - 1) / p.G;
    p.G = (p.NI + ngmax - 1) / ngmax;                 // no more CTAs than that many groups each need (N = 2048, FP32: 128 x 4, not 68 x 3 + 80 x 4)
    p.nbmax = ngmax * IB;
    p.JS = 1;
    while (ngmax * p.JS * 2 <= LEAN_NW && N / (p.JS * 2) >= 64) p.JS *= 2;
    p.JL = (((N + p.JS - 1) / p.JS) + 31) & ~31;
    p.npart = ngmax * p.JS * IB * 3;
    if (p.npart < 4 * LEAN_NW) p.npart = 4 * LEAN_NW;
    p.smem = f32 ? lean_smem_bytes<true>(N, p.npart, p.nbmax) : lean_smem_bytes<false>(N, p.npart, p.nbmax);
    p.fn = f32 ? (const void*)lean_kernel<true> : (const void*)lean_kernel<false>;
    return p;
}

}  // namespace

// CTAs the small-system kernel may use for this handle (one per SM), 0 if it cannot run: N too large for the
// shared memory of an SM or for one owner thread per body.
int lean_max_blocks(const Handle* h, int precision)
{
    if (h->N < 1 || h->N > LEAN_NMAX || 8 * h->num_sms > LEAN_SLOTW) return 0;
    const int blocks = h->num_sms;
    const LeanPlan p = lean_plan(h->N, precision, blocks);
    if (p.nbmax > LEAN_NT) return 0;
    // mergers only lower N: this N's opt-in covers every later launch
    if (cudaFuncSetAttribute(p.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(p.smem + 256)) != cudaSuccess) { cudaGetLastError(); return 0; }
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, p.fn, LEAN_NT, p.smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    if (occ < 1) return 0;
    return blocks;
}

// [v += tau_prev a] then `lead` times K and n_sds times [S D S K] (the closing velocity update left to the caller).
// The accelerations of the last evaluation are left in w.a2: the caller exchanges w.a and w.a2.
cudaError_t launch_lean(const Handle* h, const PrepArgs& prep, int precision, int lead, int n_sds, int pend,
                        double tau_prev, double tau_first, double tau_mid, double dt, int max_blocks, unsigned long long seq0)
{
    const LeanPlan p = lean_plan(h->N, precision, max_blocks);
    LeanArgs L;
    L.prep = prep; L.prep.scaled = 0;
    L.nfp = nf::make_nf_params(h);
    L.lead = lead; L.n_sds = n_sds; L.pend = pend;
    L.tau_prev = tau_prev; L.tau_first = tau_first; L.tau_mid = tau_mid;
    L.dt = dt; L.mu = h->p.G * h->p.M_star;
    L.aout = h->w.a2;
    L.seq0 = seq0;
    L.NI = p.NI; L.JS = p.JS; L.JL = p.JL; L.npart = p.npart; L.nbmax = p.nbmax;
    Workspace ws = h->w;
    cudaError_t e = cudaMemsetAsync(&h->w.ctr->pair_count, 0, sizeof(unsigned int), h->stream);
    if (e != cudaSuccess) return e;
    void* params[] = {&L, &ws};
    return cudaLaunchCooperativeKernel(p.fn, dim3((unsigned int)p.G), dim3(LEAN_NT), params, p.smem, h->stream);
}

int lean_nmax_limit() { return LEAN_NMAX; }

}  // namespace genga
