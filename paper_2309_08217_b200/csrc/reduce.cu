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

// Pair potential sum_{i<j} G m_i m_j / r_ij over the upper triangle of 128 x 128 tiles.  The tile
// pairs (ti <= tj), linearised row by row, are split evenly over the blocks; a thread holds one
// i-body of the current row tile and walks the j-tile in shared memory (four independent chains).
// TP2 mode: only pairs with i < n_big or j < n_big count (reading R9); tile pairs without any are
// skipped.  Block b writes red[8 + b]; fixed assignment and order: bitwise reproducible.
__device__ __forceinline__ void tile_of(long long u, int T, int& ti, int& tj)
{
    // row ti starts at S(ti) = ti T - ti (ti - 1) / 2; invert with a float guess, then correct
    const double B = 2.0 * T + 1.0;
    int t = (int)((B - sqrt(fmax(B * B - 8.0 * (double)u, 0.0))) * 0.5);
    if (t < 0) t = 0;
    if (t > T - 1) t = T - 1;
    while (t > 0 && (long long)t * T - (long long)t * (t - 1) / 2 > u) --t;
    while (t < T - 1 && (long long)(t + 1) * T - (long long)(t + 1) * t / 2 <= u) ++t;
    ti = t;
    tj = t + (int)(u - ((long long)t * T - (long long)t * (t - 1) / 2));
}

__global__ void __launch_bounds__(ET, 8)
pairpot_kernel(int N, int T, double G, int n_big, const double* __restrict__ x, const double* __restrict__ m,
               double* __restrict__ red)
{
    __shared__ double4 sj[ET];
    __shared__ double sh[32];
    const int tid = threadIdx.x;
    const long long U = (long long)T * (T + 1) / 2;
    const long long u0 = U * blockIdx.x / gridDim.x, u1 = U * (blockIdx.x + 1) / gridDim.x;
    double part = 0.0;
    int ti = -1, tj = 0, i = 0;
    double xi = 0, yi = 0, zi = 0, mi = 0;
    for (long long u = u0; u < u1; ++u) {
        int nti, ntj;
        if (ti < 0 || tj + 1 >= T) tile_of(u, T, nti, ntj); else { nti = ti; ntj = tj + 1; }
        if (nti != ti) {
            ti = nti; i = ti * ET + tid;
            xi = x[3 * i]; yi = x[3 * i + 1]; zi = x[3 * i + 2];
            mi = (i < N) ? m[i] : 0.0;
        }
        tj = ntj;
        if (ti * ET >= n_big && tj * ET >= n_big) continue;          // TP2: no interacting pair in this tile pair
        __syncthreads();
        {
            const int j = tj * ET + tid;
            sj[tid] = make_double4(x[3 * j], x[3 * j + 1], x[3 * j + 2], G * m[j]);
        }
        __syncthreads();
        const int jbase = tj * ET;
        const bool plain = (tj > ti) && (jbase + ET <= n_big || ti * ET + ET <= n_big);   // every pair counts
        double p0 = 0.0, p1 = 0.0, p2 = 0.0, p3 = 0.0;
        if (plain) {
#pragma unroll 2
            for (int jj = 0; jj < ET; jj += 4) {
                const double4 J0 = sj[jj], J1 = sj[jj + 1], J2 = sj[jj + 2], J3 = sj[jj + 3];
                double dx, dy, dz;
                dx = J0.x - xi; dy = J0.y - yi; dz = J0.z - zi; p0 = fma(J0.w, rsqrt_refined(fma(dz, dz, fma(dy, dy, dx * dx))), p0);
                dx = J1.x - xi; dy = J1.y - yi; dz = J1.z - zi; p1 = fma(J1.w, rsqrt_refined(fma(dz, dz, fma(dy, dy, dx * dx))), p1);
                dx = J2.x - xi; dy = J2.y - yi; dz = J2.z - zi; p2 = fma(J2.w, rsqrt_refined(fma(dz, dz, fma(dy, dy, dx * dx))), p2);
                dx = J3.x - xi; dy = J3.y - yi; dz = J3.z - zi; p3 = fma(J3.w, rsqrt_refined(fma(dz, dz, fma(dy, dy, dx * dx))), p3);
            }
        } else {
#pragma unroll 4
            for (int jj = 0; jj < ET; ++jj) {
                const double4 J = sj[jj];
                const int j = jbase + jj;
                const double dx = J.x - xi, dy = J.y - yi, dz = J.z - zi;
                const double y  = rsqrt_refined(fma(dz, dz, fma(dy, dy, dx * dx)));
                p0 = (j > i && (i < n_big || j < n_big)) ? fma(J.w, y, p0) : p0;
            }
        }
        part = fma(mi, (p0 + p1) + (p2 + p3), part);
    }
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
    long long want = (long long)T * (T + 1) / 2;
    int nblk = h->num_sms * 16;
    if (nblk > 4096) nblk = 4096;                        // partials red[8 .. 8 + 4096)
    if (nblk > want) nblk = (int)want;
    if (nblk > 0)
        pairpot_kernel<<<nblk, ET, 0, h->stream>>>(h->N, T, h->p.G, (h->p.n_big >= 0 && h->p.n_big < h->N) ? h->p.n_big : h->N,
                                                   h->w.x, h->w.m, h->w.red);
    energy_final_kernel<<<1, 1024, 0, h->stream>>>(h->N, nblk, h->p.G, h->p.M_star, h->w.m, h->w.x, h->w.v, h->w.red);
}

}  // namespace genga
