// reduce.cu -- total energy and angular momentum of the stored state (PAPER.md:111:
// "Delta E/E = E(t)/E(0) - 1 ... and likewise for L"; reading G5 / O11):
//   E = sum m v^2/2 + |sum m v|^2/(2 M_star) - sum G M_star m / r - sum_{i<j} G m_i m_j / r_ij
//   L = sum m x cross v      (democratic variables: heliocentric x, barycentric v)
// The O(N^2/2) pair potential runs as an FP64 tile loop with warp-shuffle and block reductions;
// per-block partials are combined in a fixed order (bitwise reproducible).
#include "genga_internal.cuh"

namespace genga {

namespace {

constexpr int ET = 128;      // bodies per energy tile = threads per block

__device__ __forceinline__ double rsq64h(double a)
{
    double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r;
}

// 1/sqrt(r2): MUFU.RSQ64H seed + one cubic correction, y = y0 (1 + e/2 + 3 e^2/8), e = 1 - r2 y0^2
__device__ __forceinline__ double rsqrt_refined(double r2)
{
    const double y0 = rsq64h(r2);
    const double e  = fma(-r2, y0 * y0, 1.0);
    const double p  = fma(0.375, e, 0.5);
    return fma(y0 * e, p, y0);
}

__device__ __forceinline__ double block_sum(double v, double* sh)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    const int nw = blockDim.x >> 5;
    double t = 0.0;
    if (wid == 0) {
        t = (lane < nw) ? sh[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    return t;    // valid in thread 0
}

// Block b owns i-tiles b and T-1-b (equal total work for every block): sum over j > i of
// G m_j / r_ij, times m_i, summed over the block -> red[8 + b].
__global__ void __launch_bounds__(ET)
pairpot_kernel(int N, int T, double G, int n_big, const double* __restrict__ x, const double* __restrict__ m,
               double* __restrict__ red)
{
    __shared__ double4 sj[ET];
    __shared__ double sh[32];
    const int tid = threadIdx.x;
    const int tA = blockIdx.x, tB = T - 1 - blockIdx.x;
    const int iA = tA * ET + tid, iB = tB * ET + tid;
    const bool hasB = tB > tA;
    const int iBB = hasB ? iB : iA;
    const double4 qA = make_double4(x[3 * iA], x[3 * iA + 1], x[3 * iA + 2], 0.0);
    const double4 qB = make_double4(x[3 * iBB], x[3 * iBB + 1], x[3 * iBB + 2], 0.0);
    double potA = 0.0, potB = 0.0;

    for (int tj = tA; tj < T; ++tj) {
        __syncthreads();
        {
            const int j = tj * ET + tid;
            sj[tid] = make_double4(x[3 * j], x[3 * j + 1], x[3 * j + 2], G * m[j]);
        }
        __syncthreads();
        const bool doB = hasB && tj >= tB;
        const int jbase = tj * ET;
#pragma unroll 4
        for (int jj = 0; jj < ET; ++jj) {
            const double4 J = sj[jj];
            const int j = jbase + jj;
            {
                const double dx = J.x - qA.x, dy = J.y - qA.y, dz = J.z - qA.z;
                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                const double y  = rsqrt_refined(r2);
                potA = (j > iA && (iA < n_big || j < n_big)) ? fma(J.w, y, potA) : potA;   // TP2: interacting pairs only
            }
            if (doB) {
                const double dx = J.x - qB.x, dy = J.y - qB.y, dz = J.z - qB.z;
                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                const double y  = rsqrt_refined(r2);
                potB = (j > iB && (iB < n_big || j < n_big)) ? fma(J.w, y, potB) : potB;
            }
        }
    }
    double part = 0.0;
    if (iA < N) part += m[iA] * potA;
    if (hasB && iB < N) part += m[iB] * potB;
    const double tot = block_sum(part, sh);
    if (tid == 0) red[8 + blockIdx.x] = tot;
}

// red[0] = E, red[1..3] = L.  One block; combines the O(N) sums with the pair-potential partials.
__global__ void __launch_bounds__(1024)
energy_final_kernel(int N, int nparts, double G, double M_star, const double* __restrict__ m,
                    const double* __restrict__ x, const double* __restrict__ v, double* __restrict__ red)
{
    __shared__ double sh[32];
    double kin = 0, sol = 0, p0 = 0, p1 = 0, p2 = 0, l0 = 0, l1 = 0, l2 = 0, pot = 0;
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        const double mi = m[i];
        const double X = x[3 * i], Y = x[3 * i + 1], Z = x[3 * i + 2];
        const double VX = v[3 * i], VY = v[3 * i + 1], VZ = v[3 * i + 2];
        kin = fma(0.5 * mi, fma(VZ, VZ, fma(VY, VY, VX * VX)), kin);
        sol += G * M_star * mi / sqrt(fma(Z, Z, fma(Y, Y, X * X)));
        p0 = fma(mi, VX, p0); p1 = fma(mi, VY, p1); p2 = fma(mi, VZ, p2);
        l0 = fma(mi, Y * VZ - Z * VY, l0);
        l1 = fma(mi, Z * VX - X * VZ, l1);
        l2 = fma(mi, X * VY - Y * VX, l2);
    }
    for (int b = threadIdx.x; b < nparts; b += blockDim.x) pot += red[8 + b];
    kin = block_sum(kin, sh); sol = block_sum(sol, sh); pot = block_sum(pot, sh);
    p0 = block_sum(p0, sh); p1 = block_sum(p1, sh); p2 = block_sum(p2, sh);
    l0 = block_sum(l0, sh); l1 = block_sum(l1, sh); l2 = block_sum(l2, sh);
    if (threadIdx.x == 0) {
        red[0] = kin + (p0 * p0 + p1 * p1 + p2 * p2) / (2.0 * M_star) - sol - pot;
        red[1] = l0; red[2] = l1; red[3] = l2;
    }
}

}  // namespace

// Reads x and m directly (padding bodies carry m = 0 far away), so it never disturbs the
// arrays of the last force evaluation.
void launch_energy(const Handle* h)
{
    const int T = h->NP / ET;
    const int nblk = (T + 1) / 2;
    if (nblk > 0)
        pairpot_kernel<<<nblk, ET, 0, h->stream>>>(h->N, T, h->p.G, (h->p.n_big >= 0 && h->p.n_big < h->N) ? h->p.n_big : h->N,
                                                   h->w.x, h->w.m, h->w.red);
    energy_final_kernel<<<1, 1024, 0, h->stream>>>(h->N, nblk, h->p.G, h->p.M_star, h->w.m, h->w.x, h->w.v, h->w.red);
}

}  // namespace genga
