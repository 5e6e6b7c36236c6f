// nearfield.cu -- FP64 evaluation of the (body, j-chunk) candidates the all-pairs kernels set
// aside: the changeover-weighted force (forces during an encounter "always
// calculated in double precision using changeover functions"; reading G1 for K) and the
// close-encounter pair list {(i,j): i<j, r_ij < r_crit,ij}, compacted with
// __ballot_sync + one atomic per warp.
//
// One warp per candidate, two j-bodies per lane.  Plain sqrt/divide/cbrt: this path is rare
// (about N + 2 x near pairs candidates) and must be exact.  If the candidate list overflowed,
// the kernel instead evaluates EVERY pair this way (one warp per body, overwriting a_i), so the
// result never depends on the capacity.
#include "genga_internal.cuh"

namespace genga {

namespace {

struct NfParams {
    int N, nchunk;
    double M_star, n1, n2dt;
    int pair_rule;
    unsigned int cand_cap, pair_cap;
};

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

// O4: K(r, r_crit), reading G1 (Chambers-1999 rational form)
__device__ __forceinline__ double changeover(double r, double rc)
{
    if (!(rc > 0.0)) return (r > 0.0) ? 1.0 : 0.0;
    const double y = (r - 0.1 * rc) / (0.9 * rc);
    if (y <= 0.0) return 0.0;
    if (y >= 1.0) return 1.0;
    return (y * y) / (2.0 * y * y - 2.0 * y + 1.0);
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

// force of chunk c on body i, summed over the warp; lanes return the same total
__device__ __forceinline__ void chunk_on_body(const NfParams& P, Workspace& w, int i, int c,
                                              double xi, double yi, double zi, double mi, double rci,
                                              double ai, double vki, double& fx, double& fy, double& fz)
{
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int h = 0; h < CHUNK / 32; ++h) {
        const int j = c * CHUNK + h * 32 + lane;
        double sx = 0.0, sy = 0.0, sz = 0.0;
        bool enc = false;
        if (j < P.N && j != i) {
            const double4 q = w.pk64[j];
            const double dx = q.x - xi, dy = q.y - yi, dz = q.z - zi;
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double r  = sqrt(r2);
            const double rc = pair_rcrit(P, mi, w.m[j], rci, w.rcrit[j], ai, w.semi[j], vki, w.vkep[j]);
            enc = (i < j) && (r < rc);                     // coincident bodies (r = 0) are an encounter
            if (r > 0.0) {
                const double W = changeover(r, rc);
                if (W != 0.0) {
                    const double s = q.w * W / (r2 * r);
                    sx = s * dx; sy = s * dy; sz = s * dz;
                }
            }
        }
        append_pair(enc, i, j, w, P.pair_cap);
        fx += sx; fy += sy; fz += sz;
    }
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__global__ void __launch_bounds__(128)
nearfield_kernel(NfParams P, Workspace w)
{
    const int lane  = threadIdx.x & 31;
    const int warp  = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarp = (gridDim.x * blockDim.x) >> 5;
    const unsigned int count = w.ctr->cand_count;

    if (count <= P.cand_cap) {
        for (unsigned int q = warp; q < count; q += nwarp) {
            const int2 cd = w.cand[q];
            const int i = cd.x, c = cd.y;
            const double4 pi = w.pk64[i];
            double fx = 0.0, fy = 0.0, fz = 0.0;
            chunk_on_body(P, w, i, c, pi.x, pi.y, pi.z, w.m[i], w.rcrit[i], w.semi[i], w.vkep[i], fx, fy, fz);
            fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
            if (lane == 0) {
                atomicAdd(&w.a[3 * i + 0], fx);
                atomicAdd(&w.a[3 * i + 1], fy);
                atomicAdd(&w.a[3 * i + 2], fz);
            }
        }
    } else {
        // exact slow path: the candidate list overflowed, redo every body against every chunk
        if (warp == 0 && lane == 0) w.ctr->overflow = 1u;
        for (int i = warp; i < P.N; i += nwarp) {
            const double4 pi = w.pk64[i];
            const double mi = w.m[i], rci = w.rcrit[i], ai = w.semi[i], vki = w.vkep[i];
            double fx = 0.0, fy = 0.0, fz = 0.0;
            for (int c = 0; c < P.nchunk; ++c)
                chunk_on_body(P, w, i, c, pi.x, pi.y, pi.z, mi, rci, ai, vki, fx, fy, fz);
            fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
            if (lane == 0) { w.a[3 * i + 0] = fx; w.a[3 * i + 1] = fy; w.a[3 * i + 2] = fz; }
        }
    }
}

}  // namespace

void launch_nearfield(const Handle* h)
{
    if (h->N == 0) return;
    NfParams P;
    P.N = h->N; P.nchunk = (h->N + CHUNK - 1) / CHUNK;
    P.M_star = h->p.M_star; P.n1 = h->p.n1; P.n2dt = h->p.n2 * h->p.dt_rcrit;
    P.pair_rule = h->p.pair_rule;
    P.cand_cap = (unsigned int)h->cand_cap; P.pair_cap = (unsigned int)h->pair_cap;
    int blocks = h->num_sms * 8;
    const long long need = ((long long)h->N + 3) / 4;            // at least one warp per body is enough
    if (blocks > need && need > 0) blocks = (int)((need < h->num_sms) ? h->num_sms : need);
    nearfield_kernel<<<blocks, 128, 0, h->stream>>>(P, h->w);
}

}  // namespace genga
