// onbody_body.cuh -- the O(N) rows of the step around the all-pairs kick in ONE cooperative kernel:
//   phase 1  v_i += tau_v a_i (row a6, closing the previous kick)      and  P  = sum m v   (grid-wide)
//   phase 2  x_i += (dt/2) P / M_star (row a7, Sun-kick, reading G3), Kepler drift D(dt) (row a8,
//            always FP64)                                  and  P' = sum m v'  (grid-wide)
//            [ENC: the bodies of an encounter group are advanced by one warp per group instead, encounter.cuh]
//   phase 3  x_i += (dt/2) P' / M_star, then r_crit (Eq. 1), packing and bounds (rows a1, a2) for the
//            next force evaluation.
// Each phase is optional.  The two grid-wide sums are block partials combined by EVERY block in the
// same fixed order after a grid.sync(), so all blocks hold bitwise the same P (and the result is
// reproducible for a given grid).  A step is then 3 launches: this kernel, the all-pairs kernel,
// the near-field kernel.
#pragma once

#include <cooperative_groups.h>

#include "genga_internal.cuh"
#include "encounter.cuh"
#include "kepler.cuh"
#include "momentum.cuh"
#include "prep_tile.cuh"

namespace genga {
namespace ob {

namespace cg = cooperative_groups;


constexpr int FUSED_NT = PREP_NT;          // 256: prep_tile needs exactly this block size

// Sum of the per-block partials part[4 b + k], b < nblk, by one warp with a fixed assignment and tree.
__device__ __forceinline__ void combine_partials(const double* __restrict__ part, int nblk, double* s_out)
{
    if (threadIdx.x < 32) {
        double p0 = 0, p1 = 0, p2 = 0, mt = 0;
        for (int b = threadIdx.x; b < nblk; b += 32) {
            const double* q = part + 4 * b;
            p0 += __ldcg(q + 0); p1 += __ldcg(q + 1); p2 += __ldcg(q + 2); mt += __ldcg(q + 3);
        }
        warp_sum4(p0, p1, p2, mt);
        if (threadIdx.x == 0) { s_out[0] = p0; s_out[1] = p1; s_out[2] = p2; s_out[3] = mt; }
    }
    __syncthreads();
}

// block partial of (p0, p1, p2, mt) -> part[4 blockIdx.x ..]
__device__ __forceinline__ void block_partial(double p0, double p1, double p2, double mt, double* __restrict__ part)
{
    __shared__ double s_w[FUSED_NT / 32][4];
    warp_sum4(p0, p1, p2, mt);
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { s_w[wid][0] = p0; s_w[wid][1] = p1; s_w[wid][2] = p2; s_w[wid][3] = mt; }
    __syncthreads();
    if (wid == 0) {
        const bool in = lane < FUSED_NT / 32;
        p0 = in ? s_w[lane][0] : 0.0; p1 = in ? s_w[lane][1] : 0.0; p2 = in ? s_w[lane][2] : 0.0; mt = in ? s_w[lane][3] : 0.0;
        warp_sum4(p0, p1, p2, mt);
        if (lane == 0) {
            double* q = part + 4 * blockIdx.x;
            __stcg(q + 0, p0); __stcg(q + 1, p1); __stcg(q + 2, p2); __stcg(q + 3, mt);
        }
    }
    __syncthreads();
}

// The kernel as a device function (a cooperative 1-D grid of FUSED_NT-thread blocks).
// ENC: 0 no encounter groups, 1 groups by Bulirsch-Stoer / RK4 (two-level step), 2 also in-drift collisions and sub-levels
template <int CHUNK, int ENC = 0>
__device__ __forceinline__ void onbody_body(const OnBodyArgs& A, Workspace& w, cg::grid_group& grid)
{
    __shared__ double sP[4];
    const int N = A.prep.N;
    const int gtid = blockIdx.x * FUSED_NT + threadIdx.x, gsz = gridDim.x * FUSED_NT;
    double* part1 = w.mom + MOM_PARTIALS;
    double* part2 = part1 + 4 * MOM_MAX_BLOCKS;

    // ---- phase 1: close the previous kick, total momentum of the stored velocities ----------------
    if (A.do_drift && A.reuse_P) {
        // reading R17: a kick does not change the total momentum (reciprocal pair forces), so sum m v of the velocities this
        // phase produces is the sum m v' the previous drift left in slot B: no sum, no grid-wide barrier.  (Each thread
        // updates and later drifts the same bodies i = gtid + k gsz: no other ordering is needed.)
        if (A.do_vel)
            for (int i = gtid; i < N; i += gsz) {
                w.v[3 * i + 0] = fma(A.tau_v, w.a[3 * i + 0], w.v[3 * i + 0]); w.v[3 * i + 1] = fma(A.tau_v, w.a[3 * i + 1], w.v[3 * i + 1]);
                w.v[3 * i + 2] = fma(A.tau_v, w.a[3 * i + 2], w.v[3 * i + 2]);
            }
        if (threadIdx.x < 4) sP[threadIdx.x] = w.mom[MOM_SLOT_B + threadIdx.x];
        __syncthreads();
    } else {
        double p0 = 0, p1 = 0, p2 = 0, mt = 0;
        for (int i = gtid; i < N; i += gsz) {
            double v0 = w.v[3 * i + 0], v1 = w.v[3 * i + 1], v2 = w.v[3 * i + 2];
            if (A.do_vel) {
                v0 = fma(A.tau_v, w.a[3 * i + 0], v0); v1 = fma(A.tau_v, w.a[3 * i + 1], v1); v2 = fma(A.tau_v, w.a[3 * i + 2], v2);
                w.v[3 * i + 0] = v0; w.v[3 * i + 1] = v1; w.v[3 * i + 2] = v2;
            }
            const double mi = w.m[i];
            p0 = fma(mi, v0, p0); p1 = fma(mi, v1, p1); p2 = fma(mi, v2, p2); mt += mi;
        }
        block_partial(p0, p1, p2, mt, part1);
        grid.sync();
        combine_partials(part1, gridDim.x, sP);
        if (blockIdx.x == 0 && threadIdx.x < 4) w.mom[MOM_SLOT_A + threadIdx.x] = sP[threadIdx.x];
    }
    double shx = 0.0, shy = 0.0, shz = 0.0;
    bool pending = false;

    // ---- phase 2: Sun-kick, Kepler drift, momentum of the drifted velocities --------------------------
    if (A.do_drift) {
        const double sc = 0.5 * A.dt / A.prep.M_star;
        const double s0 = sc * sP[0], s1 = sc * sP[1], s2 = sc * sP[2];
        __syncthreads();                                   // sP is rewritten below
        double p0 = 0, p1 = 0, p2 = 0, mt = 0;
        for (int i = gtid; i < N; i += gsz) {
            if (ENC) { if (w.glabel[i] >= 0) continue; }   // bodies of an encounter group: moved by their group's warp
            double x0 = w.x[3 * i] + s0, y0 = w.x[3 * i + 1] + s1, z0 = w.x[3 * i + 2] + s2;
            double vx = w.v[3 * i], vy = w.v[3 * i + 1], vz = w.v[3 * i + 2];
            if (A.dt != 0.0) {
                if (!kepler_drift(A.mu, A.dt, x0, y0, z0, vx, vy, vz)) atomicAdd(&w.ctr->noconv, 1u);
                w.v[3 * i] = vx; w.v[3 * i + 1] = vy; w.v[3 * i + 2] = vz;
            }
            w.x[3 * i] = x0; w.x[3 * i + 1] = y0; w.x[3 * i + 2] = z0;
            const double mi = w.m[i];
            p0 = fma(mi, vx, p0); p1 = fma(mi, vy, p1); p2 = fma(mi, vz, p2); mt += mi;
        }
        if (ENC) {
            // encounter mode (NEXT-1, encounter.cuh): one team (a warp, or the CTA for a large group) per encounter group
            // advances its members through the same S(dt/2) and the flow of H_A,group over dt; then their m v' joins the sum, each body's in the
            // thread that owns the body (so the sum does not depend on which warp moved which group)
            __shared__ enc::EncSmem esm;
            __shared__ int s_big[64], s_nbig;
            const int ngroups = (int)__ldcg(&w.ctr->enc_groups);
            // groups of more than enc::WMAX bodies first, each by a whole CTA (group g by CTA g mod grid).  Only if there is
            // one (group_kernel leaves the largest size): walking the group table costs a dependent global load per group
            // and CTA (430 groups: 0.25 ms, which used to be most of the hybrid step's drift).  The CTA's threads look at
            // its groups together and queue the large ones (in runs of 64).
            if ((int)__ldcg(&w.ctr->enc_maxsize) > enc::WMAX) {
                for (int g0 = (int)blockIdx.x; g0 < ngroups; g0 += 64 * (int)gridDim.x) {
                    if (threadIdx.x == 0) s_nbig = 0;
                    __syncthreads();
                    if (threadIdx.x < 64) {
                        const int g = g0 + (int)threadIdx.x * (int)gridDim.x;
                        if (g < ngroups && __ldcg(&w.ginfo[2 * g + 1]) > enc::WMAX) s_big[atomicAdd(&s_nbig, 1)] = g;
                    }
                    __syncthreads();
                    const int nb = s_nbig;
                    for (int q = 0; q < nb; ++q) {
                        int n;
                        const int* mem = enc::group_members(w, A.enc.maxgroups, s_big[q], n);
                        enc::block_group<(ENC > 1)>(A.enc, w, esm.b, mem, n, A.dt, s0, s1, s2);
                        __syncthreads();
                    }
                }
            }
            __syncthreads();
            // the others by one warp each: group g -> block g % gridDim.x, warp (g / gridDim.x) % 8
            for (int g = blockIdx.x + gridDim.x * (threadIdx.x >> 5); g < ngroups; g += gridDim.x * (FUSED_NT / 32)) {
                int n;
                const int* mem = enc::group_members(w, A.enc.maxgroups, g, n);
                if (n <= enc::WMAX) enc::warp_group<(ENC > 1)>(A.enc, w, esm.w[threadIdx.x >> 5], mem, n, A.dt, s0, s1, s2);
            }
            grid.sync();
            for (int i = gtid; i < N; i += gsz)
                if (w.glabel[i] >= 0) {
                    const double mi = w.m[i];
                    p0 = fma(mi, __ldcg(&w.v[3 * i]), p0); p1 = fma(mi, __ldcg(&w.v[3 * i + 1]), p1);
                    p2 = fma(mi, __ldcg(&w.v[3 * i + 2]), p2); mt += mi;
                }
        }
        block_partial(p0, p1, p2, mt, part2);
        grid.sync();
        combine_partials(part2, gridDim.x, sP);
        if (blockIdx.x == 0 && threadIdx.x < 4) w.mom[MOM_SLOT_B + threadIdx.x] = sP[threadIdx.x];
        shx = sc * sP[0]; shy = sc * sP[1]; shz = sc * sP[2];
        pending = true;
    }

    // ---- phase 3: closing Sun-kick, r_crit, packing, bounds ------------------------------------------------
    if (A.do_prep) {
        const int ntile = A.prep.NP / PREP_NT;
        for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x)
            prep_tile<CHUNK>(A.prep, w, tile, pending, shx, shy, shz);
    } else if (pending) {
        for (int i = gtid; i < N; i += gsz) { w.x[3 * i] += shx; w.x[3 * i + 1] += shy; w.x[3 * i + 2] += shz; }
    }
}

}  // namespace ob
}  // namespace genga
