// momentum.cuh -- grid-wide sum of m_i v_i (and of m_i) as the epilogue of an O(N) kernel:
// every block reduces its threads' terms to a partial; the last block to finish (ticket) combines
// the partials with a fixed assignment and tree, so the result is bitwise reproducible for a
// given grid.  Used by the Sun-kick (reading G3: x_i += tau sum_j m_j v_j / M_star).
#pragma once

#include "genga_internal.cuh"

namespace genga {

constexpr int MOM_SLOT_A = 0;     // mom[0..3]: sum m v (x, y, z) and sum m of the stored velocities
constexpr int MOM_SLOT_B = 4;     // mom[4..7]: the same after the last fused drift
constexpr int MOM_PARTIALS = 8;   // mom[8 + 4 b ..]: per-block partials

__device__ __forceinline__ void warp_sum4(double& a, double& b, double& c, double& d)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o); b += __shfl_down_sync(0xffffffffu, b, o);
        c += __shfl_down_sync(0xffffffffu, c, o); d += __shfl_down_sync(0xffffffffu, d, o);
    }
}

// Must be called by every thread of every block (blockDim.x a multiple of 32, at most 1024).
// out[0..3] receives the grid total once the last block is done.
__device__ __forceinline__ void grid_momentum(double p0, double p1, double p2, double mt,
                                              double* __restrict__ partials, double* __restrict__ out,
                                              unsigned int* __restrict__ ticket)
{
    __shared__ double s_part[32][4];
    __shared__ bool s_last;
    warp_sum4(p0, p1, p2, mt);
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    if (lane == 0) { s_part[wid][0] = p0; s_part[wid][1] = p1; s_part[wid][2] = p2; s_part[wid][3] = mt; }
    __syncthreads();
    if (wid == 0) {
        const bool in = lane < nw;
        p0 = in ? s_part[lane][0] : 0.0; p1 = in ? s_part[lane][1] : 0.0;
        p2 = in ? s_part[lane][2] : 0.0; mt = in ? s_part[lane][3] : 0.0;
        warp_sum4(p0, p1, p2, mt);
        if (lane == 0) {
            double* q = partials + 4 * blockIdx.x;
            q[0] = p0; q[1] = p1; q[2] = p2; q[3] = mt;
            __threadfence();
            s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
        }
    }
    __syncthreads();
    if (!s_last || wid != 0) return;
    __threadfence();
    p0 = p1 = p2 = mt = 0.0;
    for (int b = lane; b < (int)gridDim.x; b += 32) {
        const volatile double* q = partials + 4 * b;
        p0 += q[0]; p1 += q[1]; p2 += q[2]; mt += q[3];
    }
    warp_sum4(p0, p1, p2, mt);
    if (lane == 0) { out[0] = p0; out[1] = p1; out[2] = p2; out[3] = mt; *ticket = 0u; }
}

}  // namespace genga
