// noalloc.cu -- genga_energy_angmom_static: E and L of a state (O11; the arithmetic of reduce.cu)
// for callers that cannot allocate: no handle, no workspace, no cudaMalloc / cudaFree / allocating library call.
//
// The handle's path (reduce.cu) reads the padded arrays of its workspace and leaves the per-block partials of the
// O(N^2/2) pair potential in the workspace's scratch.  This variant takes the caller's plain arrays of N bodies and
// keeps BOTH in one file-scope device array of a fixed size: the bodies packed as (x, y, z, G m) records, padded to
// a whole number of 128-body tiles, and the per-block partials.  The array is part of the library image: every GPU
// that loads the library holds its 4.2 MB until the process exits, and ALL calls share it.  Nothing in it has to
// start at zero -- a call rewrites every record up to its own padded size and every partial it later reads -- but
// it keeps the last call's contents, so two calls that overlap on the GPU (different streams, or different host
// threads on unordered streams) race on it.  Calls on one stream are ordered and safe.
//
// In host code `g_static_scratch` is only a stand-in for the symbol, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current (static_setup).
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/genga.h"

namespace {

constexpr int ST = 128;                                  // bodies per tile = threads per block
constexpr int S_MAXBLK = 4096;                           // most blocks of the pair-potential kernel
static_assert(GENGA_STATIC_NMAX % ST == 0, "the padded body count must fit the array");
constexpr size_t S_PK_DOUBLES = 4 * (size_t)GENGA_STATIC_NMAX;          // [NMAX] records of 4 doubles ...
constexpr size_t S_DOUBLES = S_PK_DOUBLES + S_MAXBLK;                    // ... then [S_MAXBLK] partials

static __device__ __align__(256) double g_static_scratch[S_DOUBLES];

thread_local char t_err[256] = "";

constexpr int MAXDEV = 64;
std::mutex g_mu;
double* g_ptr[MAXDEV];                                   // device address of g_static_scratch on device d (nullptr: not asked yet)
int g_sms[MAXDEV];

int fail_cuda(cudaError_t e, const char* where)
{
    std::snprintf(t_err, sizeof(t_err), "genga_energy_angmom_static: %s: %s", where, cudaGetErrorString(e));
    return GENGA_ECUDA;
}

// Once per device, with that device current: the device address of the scratch array and the SM count.
int static_setup(double** ptr, int* sms)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "cudaGetDevice");
    if (dev < 0 || dev >= MAXDEV) {
        std::snprintf(t_err, sizeof(t_err), "genga_energy_angmom_static: device ordinal %d not supported (< %d)", dev, MAXDEV);
        return GENGA_EINVAL;
    }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
        if (e != cudaSuccess || !p) return fail_cuda(e, "cudaGetSymbolAddress(g_static_scratch)");
        int n = 0;
        e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || n < 1) return fail_cuda(e, "cudaDeviceGetAttribute(MultiProcessorCount)");
        g_sms[dev] = n;
        g_ptr[dev] = p;
    }
    *ptr = g_ptr[dev];
    *sms = g_sms[dev];
    return GENGA_OK;
}

__device__ __forceinline__ double rsq64h(double a)
{
    double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r;
}

// 1/sqrt(r2): MUFU.RSQ64H seed + one cubic correction, y = y0 (1 + e/2 + 3 e^2/8), e = 1 - r2 y0^2 (as reduce.cu)
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

// Slot s < NP of the scratch: (x, y, z, G m) of body s, or, for s >= N, a massless body far away, every one at its
// own place (their mutual terms are then 0 * finite = 0).  Rewrites every record a later kernel of this call reads.
__global__ void static_pack_kernel(int N, int NP, double G, const double* __restrict__ m, const double* __restrict__ x,
                                   double4* __restrict__ pk)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= NP) return;
    if (s < N) pk[s] = make_double4(x[3 * s], x[3 * s + 1], x[3 * s + 2], G * m[s]);
    else       pk[s] = make_double4(1.0e15 + 1.0e3 * (double)(s - N + 1), 0.0, 0.0, 0.0);
}

// row ti of the upper triangle of T x T tiles starts at tile pair S(ti) = ti T - ti (ti - 1) / 2
__device__ __forceinline__ void tile_of(long long u, int T, int& ti, int& tj)
{
    const double B = 2.0 * T + 1.0;
    int t = (int)((B - sqrt(fmax(B * B - 8.0 * (double)u, 0.0))) * 0.5);
    if (t < 0) t = 0;
    if (t > T - 1) t = T - 1;
    while (t > 0 && (long long)t * T - (long long)t * (t - 1) / 2 > u) --t;
    while (t < T - 1 && (long long)(t + 1) * T - (long long)(t + 1) * t / 2 <= u) ++t;
    ti = t;
    tj = t + (int)(u - ((long long)t * T - (long long)t * (t - 1) / 2));
}

// Pair potential sum_{i<j} G m_i m_j / r_ij over the upper triangle of 128 x 128 tiles of the packed records (the
// loop of reduce.cu: pairpot_kernel without its TP2 case).  Block b writes part[b], always: nothing is accumulated
// into the shared array, so nothing of an earlier call can leak into this one.
__global__ void __launch_bounds__(ST, 8)
static_pairpot_kernel(int N, int T, const double* __restrict__ m, const double4* __restrict__ pk, double* __restrict__ part)
{
    __shared__ double4 sj[ST];
    __shared__ double sh[32];
    const int tid = threadIdx.x;
    const long long U = (long long)T * (T + 1) / 2;
    const long long u0 = U * blockIdx.x / gridDim.x, u1 = U * (blockIdx.x + 1) / gridDim.x;
    double acc = 0.0;
    int ti = -1, tj = 0, i = 0;
    double xi = 0, yi = 0, zi = 0, mi = 0;
    for (long long u = u0; u < u1; ++u) {
        int nti, ntj;
        if (ti < 0 || tj + 1 >= T) tile_of(u, T, nti, ntj); else { nti = ti; ntj = tj + 1; }
        if (nti != ti) {
            ti = nti; i = ti * ST + tid;
            const double4 q = pk[i];
            xi = q.x; yi = q.y; zi = q.z;
            mi = (i < N) ? m[i] : 0.0;
        }
        tj = ntj;
        __syncthreads();
        sj[tid] = pk[tj * ST + tid];
        __syncthreads();
        const int jbase = tj * ST;
        double p0 = 0.0, p1 = 0.0, p2 = 0.0, p3 = 0.0;
        if (tj > ti) {                                   // every pair of the tile pair counts
#pragma unroll 2
            for (int jj = 0; jj < ST; jj += 4) {
                const double4 J0 = sj[jj], J1 = sj[jj + 1], J2 = sj[jj + 2], J3 = sj[jj + 3];
                double dx, dy, dz;
                dx = J0.x - xi; dy = J0.y - yi; dz = J0.z - zi; p0 = fma(J0.w, rsqrt_refined(fma(dz, dz, fma(dy, dy, dx * dx))), p0);
                dx = J1.x - xi; dy = J1.y - yi; dz = J1.z - zi; p1 = fma(J1.w, rsqrt_refined(fma(dz, dz, fma(dy, dy, dx * dx))), p1);
                dx = J2.x - xi; dy = J2.y - yi; dz = J2.z - zi; p2 = fma(J2.w, rsqrt_refined(fma(dz, dz, fma(dy, dy, dx * dx))), p2);
                dx = J3.x - xi; dy = J3.y - yi; dz = J3.z - zi; p3 = fma(J3.w, rsqrt_refined(fma(dz, dz, fma(dy, dy, dx * dx))), p3);
            }
        } else {                                         // the tile against itself: j > i, by selection (r = 0 at j = i)
#pragma unroll 4
            for (int jj = 0; jj < ST; ++jj) {
                const double4 J = sj[jj];
                const double dx = J.x - xi, dy = J.y - yi, dz = J.z - zi;
                const double y  = rsqrt_refined(fma(dz, dz, fma(dy, dy, dx * dx)));
                p0 = (jbase + jj > i) ? fma(J.w, y, p0) : p0;
            }
        }
        acc = fma(mi, (p0 + p1) + (p2 + p3), acc);
    }
    const double tot = block_sum(acc, sh);
    if (tid == 0) part[blockIdx.x] = tot;
}

// out4 = (E, Lx, Ly, Lz).  One block; the O(N) sums of the caller's arrays and the nparts partials in a fixed order
// (reduce.cu: energy_final_kernel).
__global__ void __launch_bounds__(1024)
static_final_kernel(int N, int nparts, double G, double M_star, const double* __restrict__ m, const double* __restrict__ x,
                    const double* __restrict__ v, const double* __restrict__ part, double* __restrict__ out4)
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
    for (int b = threadIdx.x; b < nparts; b += blockDim.x) pot += part[b];
    kin = block_sum(kin, sh); sol = block_sum(sol, sh); pot = block_sum(pot, sh);
    p0 = block_sum(p0, sh); p1 = block_sum(p1, sh); p2 = block_sum(p2, sh);
    l0 = block_sum(l0, sh); l1 = block_sum(l1, sh); l2 = block_sum(l2, sh);
    if (threadIdx.x == 0) {
        out4[0] = kin + (p0 * p0 + p1 * p1 + p2 * p2) / (2.0 * M_star) - sol - pot;
        out4[1] = l0; out4[2] = l1; out4[3] = l2;
    }
}

}  // namespace

extern "C" {

int genga_energy_angmom_static(int N, const double* m, const double* x, const double* v, double G, double M_star,
                               void* stream, double* out4)
{
    t_err[0] = 0;
    if (N < 0 || !out4 || !(M_star > 0.0) || (N > 0 && (!m || !x || !v))) {
        std::snprintf(t_err, sizeof(t_err), "genga_energy_angmom_static: invalid argument (N < 0, a NULL array, or M_star <= 0)");
        return GENGA_EINVAL;
    }
    if (N > GENGA_STATIC_NMAX) {
        std::snprintf(t_err, sizeof(t_err), "genga_energy_angmom_static: N = %d exceeds GENGA_STATIC_NMAX = %d, the fixed size of "
                      "the library's static scratch array; use a handle (genga_energy_angmom) for larger systems", N, GENGA_STATIC_NMAX);
        return GENGA_ELIMIT;
    }
    double* scratch = nullptr;
    int sms = 0;
    const int rc = static_setup(&scratch, &sms);
    if (rc != GENGA_OK) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    double4* pk = reinterpret_cast<double4*>(scratch);
    double* part = scratch + S_PK_DOUBLES;
    int nblk = 0;
    if (N > 0) {
        const int NP = (N + ST - 1) / ST * ST, T = NP / ST;
        const long long want = (long long)T * (T + 1) / 2;
        nblk = sms * 16;
        if (nblk > S_MAXBLK) nblk = S_MAXBLK;
        if (nblk > want) nblk = (int)want;
        static_pack_kernel<<<NP / ST, ST, 0, s>>>(N, NP, G, m, x, pk);
        static_pairpot_kernel<<<nblk, ST, 0, s>>>(N, T, m, pk, part);
    }
    static_final_kernel<<<1, 1024, 0, s>>>(N, nblk, G, M_star, m, x, v, part, out4);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "kernel launch");
    return GENGA_OK;
}

const char* genga_static_last_error(void) { return t_err; }

}  // extern "C"
