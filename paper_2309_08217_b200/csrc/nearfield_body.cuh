// nearfield_body.cuh -- FP64 evaluation of the (body, j-chunk) candidates the all-pairs kernels set
// aside: the changeover-weighted force (forces during an encounter "always
// calculated in double precision using changeover functions"; reading G1 for K) and the
// close-encounter pair list {(i,j): i<j, r_ij < r_crit,ij}, compacted with
// __ballot_sync + one atomic per warp.
//
// One warp per candidate, four j-bodies per lane, two phases (cheap K = 1 terms; compacted near
// pairs with plain sqrt/divide/cbrt: this path is rare and must be exact).  If the candidate list overflowed,
// the kernel instead evaluates EVERY pair this way (one warp per body, overwriting a_i), so the
// result never depends on the capacity.
#pragma once

#include "genga_internal.cuh"

namespace genga {
namespace nf {


struct NfParams {
    int N, nchunk;
    double M_star, n1, n2dt;
    int pair_rule;
    int weight_mode;                               // 0: W = K, 1: W = K - r dK/dr (reading R10)
    double list_scale;                             // pairs with r < list_scale r_crit,ij are listed (1 unless encounter mode)
    double list_vdt;                               // ... and, if >= 0, only those with r - r_crit,ij < list_vdt |v_i - v_j|
    int check_missed;                              // encounter mode: count pairs inside their zone that the last drift had not grouped
    unsigned int cand_cap, pair_cap;
    int gather, NP;                                // fold aslot[] (sums of the symmetric all-pairs kernels) into a[] first
};

inline NfParams make_nf_params(const Handle* h)
{
    NfParams P;
    P.N = h->N; P.nchunk = h->nchunk;
    P.M_star = h->p.M_star; P.n1 = h->p.n1; P.n2dt = h->p.n2 * h->p.dt_rcrit;
    P.pair_rule = h->p.pair_rule; P.weight_mode = h->p.weight_mode;
    P.list_scale = (h->p.encounter_mode != 0) ? h->p.enc_list_scale : 1.0;
    P.list_vdt = (h->p.encounter_mode != 0 && h->p.enc_list_vfactor >= 0.0) ? h->p.enc_list_vfactor * h->enc_dt : -1.0;
    P.check_missed = (h->p.encounter_mode != 0 && h->enc_labels_valid) ? 1 : 0;
    P.cand_cap = (unsigned int)h->cand_cap; P.pair_cap = (unsigned int)h->pair_cap;
    P.gather = 0; P.NP = h->NP;
    return P;
}

// O3: r_crit,ij from per-body quantities (reading G2)
__device__ __forceinline__ double pair_rcrit(const NfParams& P, double mi, double mj, double rci, double rcj,
                                             double ai, double aj, double vki, double vkj)
{
    if (P.pair_rule == GENGA_PAIR_MUTUAL_HILL) {
        const double hill = P.n1 * cbrt((mi + mj) / (3.0 * P.M_star)) * (0.5 * (ai + aj));
        const double vel  = P.n2dt * fmax(vki, vkj);
        return fmax(hill, vel);
    }
    return fmax(rci, rcj);
}

// O4: pair weight W(r, r_crit).  K, reading G1 (Chambers-1999 rational form); mode 1 (reading R10):
// K - r dK/dr, the weight that makes the kick the gradient of the pair potential -G m_i m_j K / r.
__device__ __forceinline__ double changeover(double r, double rc, int mode)
{
    if (!(rc > 0.0)) return (r > 0.0) ? 1.0 : 0.0;
    const double y = (r - 0.1 * rc) / (0.9 * rc);
    if (y <= 0.0) return 0.0;
    if (y >= 1.0) return 1.0;
    const double D = 2.0 * y * y - 2.0 * y + 1.0;
    const double K = (y * y) / D;
    if (mode == 0) return K;
    return K - r * ((2.0 * y * (1.0 - y) / (D * D)) / (0.9 * rc));
}

__device__ __forceinline__ void append_pair(bool flag, int i, int j, Workspace& w, unsigned int cap)
{
    const unsigned int bal = __ballot_sync(0xffffffffu, flag);
    if (!bal) return;
    const unsigned int lane = threadIdx.x & 31u;
    const int leader = __ffs(bal) - 1;
    unsigned int base = 0;
    if ((int)lane == leader) base = atomicAdd(&w.ctr->pair_count, (unsigned int)__popc(bal));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (flag) {
        const unsigned int idx = base + __popc(bal & ((1u << lane) - 1u));
        if (idx < cap) w.pairs[idx] = make_int2(i, j);
    }
}

__device__ __forceinline__ double rsq64h(double a)
{
    double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r;
}

// what the warp holds of body (slot) si while it walks a chunk
struct IBody {
    int    slot, body;
    double x, y, z;
    double m, rc, a, vk;
    float  hq, aq, rf;
};

__device__ __forceinline__ IBody load_ibody(const Workspace& w, int si)
{
    IBody b;
    b.slot = si; b.body = w.order[si];
    const double4 p = w.pk64[si]; b.x = p.x; b.y = p.y; b.z = p.z;
    const double4 q = w.aux[si];  b.m = q.x; b.rc = q.y; b.a = q.z; b.vk = q.w;
    const BoundP bp = w.bi[si];   b.hq = bp.hq; b.aq = bp.aq; b.rf = bp.rf;
    return b;
}

// Force of chunk c on the body in slot si, partial per lane.  Two phases per (body, chunk):
//  A  every pair outside the conservative pair bound (the bound the all-pairs kernels use per
//     chunk, here per pair) has K = 1 exactly and cannot be an encounter: cheap refined-rsqrt term.
//     The slots of the other pairs are compacted (__ballot_sync) into the warp's list in shared memory.
//  B  the listed pairs, one per lane: plain sqrt / divide / cbrt, exact r < r_crit test, K, force;
//     encounter pairs appended with one atomic per warp.
// (One pass over the few near pairs with many lanes active, instead of one divergent pass per round.)
template <int CHUNK>
__device__ __forceinline__ void chunk_on_body(const NfParams& P, Workspace& w, const IBody& I, int c,
                                              int* __restrict__ near_list, double& fx, double& fy, double& fz)
{
    const int lane = threadIdx.x & 31;
    constexpr int H = CHUNK / 32;
    int nnear = 0;
#pragma unroll
    for (int h = 0; h < H; ++h) {
        const int sj = c * CHUNK + h * 32 + lane;
        bool near = false;
        if (sj < P.N && sj != I.slot) {
            const double4 q = w.pk64[sj];
            const BoundP  b = w.bi[sj];
            const double dx = q.x - I.x, dy = q.y - I.y, dz = q.z - I.z;
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            const float  Bq = fmaxf(fmaxf(I.hq, b.hq) * fmaxf(I.aq, b.aq), fmaxf(I.rf, b.rf));
            const double bd = (double)Bq * (double)Bq * 1.000001;
            near = !(r2 > bd);
            if (!near) {
                const double y0 = rsq64h(r2);
                const double t  = y0 * y0;
                const double e  = fma(-r2, t, 1.0);
                const double cc = fma(1.875, e, 1.5);
                const double g  = (q.w * y0) * t;
                const double s  = fma(g * e, cc, g);
                fx = fma(s, dx, fx); fy = fma(s, dy, fy); fz = fma(s, dz, fz);
            }
        }
        const unsigned int bal = __ballot_sync(0xffffffffu, near);
        if (near) near_list[nnear + __popc(bal & ((1u << lane) - 1u))] = sj;
        nnear += __popc(bal);
    }
    __syncwarp();
    for (int k0 = 0; k0 < nnear; k0 += 32) {
        const int k = k0 + lane;
        int encj = -1;
        if (k < nnear) {
            const int sj = near_list[k];
            const double4 q = w.pk64[sj];
            const double4 A = w.aux[sj];
            const double dx = q.x - I.x, dy = q.y - I.y, dz = q.z - I.z;
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            const double r  = sqrt(r2);
            const double rc = pair_rcrit(P, I.m, A.x, I.rc, A.y, I.a, A.z, I.vk, A.w);
            if ((I.slot < sj) && (r < P.list_scale * rc)) {                           // coincident bodies (r = 0) are an encounter
                const int bj = w.order[sj];
                bool listed = true;
                if (!(r < rc) && P.list_vdt >= 0.0) {      // encounter mode: outside the zone, listed if it can get there in a step
                    const double u0 = w.v[3 * bj] - w.v[3 * I.body], u1 = w.v[3 * bj + 1] - w.v[3 * I.body + 1],
                                 u2 = w.v[3 * bj + 2] - w.v[3 * I.body + 2];
                    listed = (r - rc) < P.list_vdt * sqrt(fma(u2, u2, fma(u1, u1, u0 * u0)));
                }
                if (listed) encj = bj;
                if (P.check_missed && (r < rc)) {          // in its zone now: was it moved as a group?
                    const int la = w.glabel[I.body], lb = w.glabel[bj];
                    if (la != -2 && lb != -2 && (la < 0 || la != lb)) atomicAdd(&w.ctr->enc_missed, 1u);
                }
            }
            if (r > 0.0) {
                const double W = changeover(r, rc, P.weight_mode);
                if (W != 0.0) {
                    const double s = q.w * W / (r2 * r);
                    fx = fma(s, dx, fx); fy = fma(s, dy, fy); fz = fma(s, dz, fz);
                }
            }
        }
        const unsigned int bal = __ballot_sync(0xffffffffu, encj >= 0);
        if (bal) {
            unsigned int base = 0;
            if (lane == 0) base = atomicAdd(&w.ctr->pair_count, (unsigned int)__popc(bal));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (encj >= 0) {
                const unsigned int idx = base + __popc(bal & ((1u << lane) - 1u));
                if (idx < P.pair_cap) w.pairs[idx] = make_int2(min(I.body, encj), max(I.body, encj));
            }
        }
    }
    __syncwarp();                                  // the list is reused by the next (body, chunk)
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// The whole near-field pass as a device function: any 1-D grid of NWARP-warp blocks.
template <int CHUNK, int NWARP>
__device__ __forceinline__ void nearfield_body(const NfParams& P, Workspace& w)
{
    __shared__ int s_near[NWARP][CHUNK];
    const int lane  = threadIdx.x & 31;
    const int warp  = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarp = (gridDim.x * blockDim.x) >> 5;
    const unsigned int count = w.ctr->cand_count;
    int* near_list = s_near[threadIdx.x >> 5];

    if (count <= P.cand_cap) {
        if (P.gather) {
            // the symmetric all-pairs kernels leave their sums in aslot[] (internal order, pairs split for coalescing):
            // a[order[s]] += aslot[s'].  Atomic, because other warps add near-field terms to the same a[] meanwhile.
            for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < P.N; s += gridDim.x * blockDim.x) {
                const int b = s & (CHUNK - 1);
                const int k = (s - b) + (b & 1) * (CHUNK / 2) + (b >> 1);
                const double vx = w.aslot[k], vy = w.aslot[P.NP + k], vz = w.aslot[2 * P.NP + k];
                if (vx != 0.0 || vy != 0.0 || vz != 0.0) {
                    const int i = w.order[s];
                    atomicAdd(&w.a[3 * i + 0], vx); atomicAdd(&w.a[3 * i + 1], vy); atomicAdd(&w.a[3 * i + 2], vz);
                }
            }
        }
        for (unsigned int q = warp; q < count; q += nwarp) {
            const int2 cd = w.cand[q];
            const IBody I = load_ibody(w, cd.x);
            double fx = 0.0, fy = 0.0, fz = 0.0;
            chunk_on_body<CHUNK>(P, w, I, cd.y, near_list, fx, fy, fz);
            fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
            if (lane == 0) {
                atomicAdd(&w.a[3 * I.body + 0], fx);
                atomicAdd(&w.a[3 * I.body + 1], fy);
                atomicAdd(&w.a[3 * I.body + 2], fz);
            }
        }
    } else {
        // exact slow path: the candidate list overflowed, redo every body against every chunk
        if (warp == 0 && lane == 0) w.ctr->overflow = 1u;
        for (int si = warp; si < P.N; si += nwarp) {
            const IBody I = load_ibody(w, si);
            double fx = 0.0, fy = 0.0, fz = 0.0;
            for (int c = 0; c < P.nchunk; ++c) chunk_on_body<CHUNK>(P, w, I, c, near_list, fx, fy, fz);
            fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
            if (lane == 0) { w.a[3 * I.body + 0] = fx; w.a[3 * I.body + 1] = fy; w.a[3 * I.body + 2] = fz; }
        }
    }
}

}  // namespace nf
}  // namespace genga
