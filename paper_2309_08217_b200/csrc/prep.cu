// prep.cu -- the O(N) kernels around the all-pairs kick: critical radius (Eq. 1),
// packing of the j-side arrays, the conservative near-field bound parameters, velocity update,
// momentum reduction, Sun-kick (reading G3) and the velocity-convention shifts (O1).
#include "genga_internal.cuh"

namespace genga {

namespace {

constexpr int PREP_NT = 256;

// cbrt(m / 3 M_star): the mass factor of the Hill radius, cached while masses are unchanged.
__global__ void hcbrt_kernel(int NP, int N, const double* __restrict__ m, double inv3M, double* __restrict__ hcbrt)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= NP) return;
    hcbrt[i] = (i < N) ? cbrt(m[i] * inv3M) : 0.0;
}

__global__ void pad_kernel(int N, int NP, double* __restrict__ m, double* __restrict__ x, double* __restrict__ v)
{
    int i = N + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= NP) return;
    m[i] = 0.0;
    x[3 * i] = PAD_POS; x[3 * i + 1] = 0.0; x[3 * i + 2] = 0.0;
    v[3 * i] = 0.0; v[3 * i + 1] = 0.0; v[3 * i + 2] = 0.0;
}

__device__ __forceinline__ unsigned int warp_max_u32(unsigned int v)
{
    return __reduce_max_sync(0xffffffffu, v);
}

// One thread per (padded) body.  Eq. 1:  r_crit,i = max(n1 R_H,i, n2 dt v_i), R_H,i = a_i (m_i/3M)^(1/3);
// a_i from vis-viva with the stored velocity (readings G2b, G2c); v_i = sqrt(G M / a_i).
__global__ void __launch_bounds__(PREP_NT)
prep_kernel(PrepArgs A, Workspace w)
{
    __shared__ unsigned int smax[PREP_NT / 32][3];
    const int i = blockIdx.x * PREP_NT + threadIdx.x;      // grid covers NP exactly (NP % 512 == 0)
    const bool live = i < A.N;

    double px = PAD_POS, py = 0.0, pz = 0.0, gm = 0.0;
    float hq = 0.f, aq = 0.f, rf = 0.f;
    if (live) {
        const double mu = A.G * A.M_star;
        px = w.x[3 * i + 0]; py = w.x[3 * i + 1]; pz = w.x[3 * i + 2];
        const double vx = w.v[3 * i + 0], vy = w.v[3 * i + 1], vz = w.v[3 * i + 2];
        const double r  = sqrt(px * px + py * py + pz * pz);
        const double v2 = vx * vx + vy * vy + vz * vz;
        double sa = 1.0 / (2.0 / r - v2 / mu);
        if (!(sa > 0.0) || !isfinite(sa)) sa = r;
        const double h  = w.hcbrt[i];
        const double vk = sqrt(mu / sa);
        const double rc = fmax(A.n1 * (sa * h), A.n2 * A.dt_rcrit * vk);
        w.rcrit[i] = rc; w.semi[i] = sa; w.vkep[i] = vk;
        gm = A.G * w.m[i];

        const double lam = (double)A.lambda * (1.0 + 1.0e-6);
        double dhq, daq, drf;
        if (A.pair_rule == GENGA_PAIR_MUTUAL_HILL) {
            dhq = lam * A.n1 * 1.2599210498948732 * h;     // cbrt(2) * h_i bounds cbrt((m_i+m_j)/3M)
            daq = sa;
            drf = fmax((double)A.floor_rel * r, lam * A.n2 * A.dt_rcrit * vk);
        } else {
            dhq = lam * rc;
            daq = 1.0;
            drf = (double)A.floor_rel * r;
        }
        hq = __double2float_ru(dhq); aq = __double2float_ru(daq); rf = __double2float_ru(drf);
        if (!(hq >= 0.f)) hq = 3.0e38f;                     // NaN state: flag everything
        if (!(aq >= 0.f)) aq = 3.0e38f;
        if (!(rf >= 0.f)) rf = 3.0e38f;
    }
    w.a[3 * i + 0] = 0.0; w.a[3 * i + 1] = 0.0; w.a[3 * i + 2] = 0.0;
    w.pk64[i] = make_double4(px, py, pz, gm);
    {
        float* f = reinterpret_cast<float*>(w.pk32) + 8 * (i >> 1) + (i & 1);
        f[0] = (float)px; f[2] = (float)py; f[4] = (float)pz; f[6] = (float)gm;
    }
    BoundP b; b.hq = hq; b.aq = aq; b.rf = rf; b.pad = live ? 1.f : 0.f;
    w.bi[i] = b;

    // per-chunk maxima (CHUNK = 64 = two warps); non-negative floats order like unsigned ints
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned int m0 = warp_max_u32(__float_as_uint(hq));
    unsigned int m1 = warp_max_u32(__float_as_uint(aq));
    unsigned int m2 = warp_max_u32(__float_as_uint(rf));
    if (lane == 0) { smax[wid][0] = m0; smax[wid][1] = m1; smax[wid][2] = m2; }
    __syncthreads();
    if (threadIdx.x < PREP_NT / CHUNK) {
        const int c = threadIdx.x;
        BoundP q;
        q.hq = __uint_as_float(max(smax[2 * c][0], smax[2 * c + 1][0]));
        q.aq = __uint_as_float(max(smax[2 * c][1], smax[2 * c + 1][1]));
        q.rf = __uint_as_float(max(smax[2 * c][2], smax[2 * c + 1][2]));
        q.pad = 0.f;
        w.bc[blockIdx.x * (PREP_NT / CHUNK) + c] = q;
    }
    if (i == 0) { w.ctr->cand_count = 0u; w.ctr->pair_count = 0u; w.ctr->overflow = 0u; }
}

// O7: v_i += tau a_i
__global__ void velupdate_kernel(int n3, double tau, const double* __restrict__ a, double* __restrict__ v)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n3) v[k] = fma(tau, a[k], v[k]);
}

// red[0..2] = sum_j m_j v_j, red[3] = sum_j m_j.  One block, fixed reduction tree (deterministic).
__global__ void __launch_bounds__(1024)
momentum_kernel(int N, const double* __restrict__ m, const double* __restrict__ v, double* __restrict__ red)
{
    __shared__ double s[32][4];
    double p0 = 0, p1 = 0, p2 = 0, mt = 0;
    for (int i = threadIdx.x; i < N; i += 1024) {
        const double mi = m[i];
        p0 = fma(mi, v[3 * i + 0], p0); p1 = fma(mi, v[3 * i + 1], p1); p2 = fma(mi, v[3 * i + 2], p2);
        mt += mi;
    }
    for (int o = 16; o > 0; o >>= 1) {
        p0 += __shfl_down_sync(0xffffffffu, p0, o); p1 += __shfl_down_sync(0xffffffffu, p1, o);
        p2 += __shfl_down_sync(0xffffffffu, p2, o); mt += __shfl_down_sync(0xffffffffu, mt, o);
    }
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { s[wid][0] = p0; s[wid][1] = p1; s[wid][2] = p2; s[wid][3] = mt; }
    __syncthreads();
    if (wid == 0) {
        p0 = s[lane][0]; p1 = s[lane][1]; p2 = s[lane][2]; mt = s[lane][3];
        for (int o = 16; o > 0; o >>= 1) {
            p0 += __shfl_down_sync(0xffffffffu, p0, o); p1 += __shfl_down_sync(0xffffffffu, p1, o);
            p2 += __shfl_down_sync(0xffffffffu, p2, o); mt += __shfl_down_sync(0xffffffffu, mt, o);
        }
        if (lane == 0) { red[0] = p0; red[1] = p1; red[2] = p2; red[3] = mt; }
    }
}

// q_i[k] += scale * red[k]: O1 (q = v, scale = -1/(M_star + sum m) with red[3], or +1/M_star) and
// O8 (q = x, scale = tau / M_star).  mode 1: scale is divided by (M_star_plus + red[3]).
__global__ void shift_kernel(int N, double scale, int mode, double M_star, const double* __restrict__ red,
                             double* __restrict__ q)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= 3 * N) return;
    double s = scale;
    if (mode == 1) s = scale / (M_star + red[3]);
    q[k] = fma(s, red[k % 3], q[k]);
}

__global__ void copy_shift_kernel(int N, double scale, const double* __restrict__ red,
                                  const double* __restrict__ v, double* __restrict__ out)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= 3 * N) return;
    out[k] = fma(scale, red[k % 3], v[k]);
}

}  // namespace

void launch_hcbrt(const Handle* h)
{
    if (h->NP == 0) return;
    hcbrt_kernel<<<(h->NP + 255) / 256, 256, 0, h->stream>>>(h->NP, h->N, h->w.m, 1.0 / (3.0 * h->p.M_star), h->w.hcbrt);
}

void launch_pad(const Handle* h)
{
    const int n = h->NP - h->N;
    if (n <= 0) return;
    pad_kernel<<<(n + 255) / 256, 256, 0, h->stream>>>(h->N, h->NP, h->w.m, h->w.x, h->w.v);
}

void launch_prep(const Handle* h, const PrepArgs& a)
{
    if (h->NP == 0) return;
    prep_kernel<<<h->NP / PREP_NT, PREP_NT, 0, h->stream>>>(a, h->w);
}

void launch_velupdate(const Handle* h, double tau)
{
    if (h->N == 0) return;
    const int n3 = 3 * h->N;
    velupdate_kernel<<<(n3 + 255) / 256, 256, 0, h->stream>>>(n3, tau, h->w.a, h->w.v);
}

void launch_momentum(const Handle* h)
{
    momentum_kernel<<<1, 1024, 0, h->stream>>>(h->N, h->w.m, h->w.v, h->w.red);
}

void launch_shift_v(const Handle* h, double scale)
{
    if (h->N == 0) return;
    const int n3 = 3 * h->N;
    // scale < 0: to democratic, v -= P/(M_star + sum m); scale > 0: to heliocentric, v += P/M_star
    if (scale < 0)
        shift_kernel<<<(n3 + 255) / 256, 256, 0, h->stream>>>(h->N, -1.0, 1, h->p.M_star, h->w.red, h->w.v);
    else
        shift_kernel<<<(n3 + 255) / 256, 256, 0, h->stream>>>(h->N, 1.0 / h->p.M_star, 0, h->p.M_star, h->w.red, h->w.v);
}

void launch_sunkick(const Handle* h, double tau)
{
    if (h->N == 0) return;
    const int n3 = 3 * h->N;
    shift_kernel<<<(n3 + 255) / 256, 256, 0, h->stream>>>(h->N, tau / h->p.M_star, 0, h->p.M_star, h->w.red, h->w.x);
}

void launch_copy_v_helio(const Handle* h, double* out)
{
    if (h->N == 0) return;
    const int n3 = 3 * h->N;
    copy_shift_kernel<<<(n3 + 255) / 256, 256, 0, h->stream>>>(h->N, 1.0 / h->p.M_star, h->w.red, h->w.v, out);
}

}  // namespace genga
