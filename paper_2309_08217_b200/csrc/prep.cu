// prep.cu -- the O(N) kernels around the all-pairs kick: critical radius (Eq. 1),
// packing of the j-side arrays, the conservative near-field bound parameters, velocity update,
// momentum reduction, Sun-kick (reading G3) and the velocity-convention shifts (O1).
#include "genga_internal.cuh"
#include "momentum.cuh"
#include "prep_tile.cuh"

namespace genga {

namespace {


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


// ---- internal order ---------------------------------------------------------------------------
// The all-pairs kernels flag (body, 64-j chunk) units with ONE conservative bound per unit, and
// the FP32 kernel works in a local frame per chunk, so a chunk should hold bodies that are alike
// and close together.  Bodies are therefore kept in an internal order: bodies much heavier than
// the mean first (their large r_crit then stays in a few chunks), then along a Hilbert curve over
// the x-y plane (the discs are thin).  The order is a performance hint only: every bound is
// computed from the actual chunk contents, so results never depend on it beyond summation order.
// key = [class:2][Hilbert index:30][body index:32], class 0 heavy, 1 ordinary, 2 massless (test particles
// last, so that they share few chunks); distinct keys, so ranks are a permutation.
constexpr int SORT_BITS = 13;                       // buckets = leading key bits: class + 12 Hilbert bits
constexpr int SORT_NB   = 1 << SORT_BITS;

__global__ void extent_kernel(int N, const double* __restrict__ x, unsigned int* __restrict__ extent_bits)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    float e = 0.f;
    if (i < N) {
        e = fmaxf(fabsf((float)x[3 * i]), fabsf((float)x[3 * i + 1]));
        if (!(e < 3.0e38f)) e = 0.f;                          // NaN / inf positions do not set the extent
    }
    const unsigned int w = __reduce_max_sync(0xffffffffu, __float_as_uint(e));
    if ((threadIdx.x & 31) == 0 && w) atomicMax(extent_bits, w);
}

// index of cell (cx, cy) of a 2^15 x 2^15 grid along the Hilbert curve (30 bits)
__device__ __forceinline__ unsigned int hilbert_xy2d(unsigned int cx, unsigned int cy)
{
    unsigned int d = 0;
    for (unsigned int s = 1u << 14; s > 0; s >>= 1) {
        const unsigned int rx = (cx & s) ? 1u : 0u, ry = (cy & s) ? 1u : 0u;
        d += s * s * ((3u * rx) ^ ry);
        if (ry == 0) {
            if (rx == 1) { cx = s - 1 - cx; cy = s - 1 - cy; }
            const unsigned int t = cx; cx = cy; cy = t;
        }
        cx &= (s - 1); cy &= (s - 1);
    }
    return d;
}

__global__ void sortkey_kernel(int N, double M_star, const double* __restrict__ x,
                               const double* __restrict__ hcbrt, const double* __restrict__ red,
                               const unsigned int* __restrict__ extent_bits, unsigned long long* __restrict__ keys,
                               unsigned int* __restrict__ hist)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float ext = fmaxf(__uint_as_float(*extent_bits), 1.0e-30f);
    const float sc  = 16383.5f / ext;                                    // [-ext, ext] -> [0, 32767]
    const float fx = fminf(fmaxf(fmaf((float)x[3 * i], sc, 16383.5f), 0.f), 32767.f);
    const float fy = fminf(fmaxf(fmaf((float)x[3 * i + 1], sc, 16383.5f), 0.f), 32767.f);
    const unsigned int cx = (fx == fx) ? (unsigned int)fx : 0u, cy = (fy == fy) ? (unsigned int)fy : 0u;
    const double href = cbrt(red[3] / ((double)N * 3.0 * M_star));      // Hill factor of the mean mass
    const double hi = hcbrt[i];
    const unsigned long long cls = (hi > 1.5 * href) ? 0ull : ((hi > 0.0) ? 1ull : 2ull);
    const unsigned long long key = (cls << 62) | ((unsigned long long)hilbert_xy2d(cx, cy) << 32) | (unsigned int)i;
    keys[i] = key;
    atomicAdd(&hist[(unsigned int)(key >> (64 - SORT_BITS))], 1u);
}

// Bucket sort on the leading SORT_BITS key bits, then exact ranks inside each bucket:
//   hist (in sortkey_kernel) -> exclusive scan -> scatter into buckets (any order) -> rank of every
//   key among the keys of its own bucket.  Keys are distinct, so the result is the exact sorted
//   order whatever order the atomics ran in.  O(N) plus O(bucket size) per body.
__global__ void __launch_bounds__(1024)
sortscan_kernel(const unsigned int* __restrict__ hist, unsigned int* __restrict__ start, unsigned int* __restrict__ cursor)
{
    __shared__ unsigned int wsum[32];
    constexpr int PER = SORT_NB / 1024;
    unsigned int v[PER], tot = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) { v[k] = hist[threadIdx.x * PER + k]; tot += v[k]; }
    unsigned int inc = tot;                                      // inclusive scan over threads
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        unsigned int w = wsum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const unsigned int t = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += t; }
        wsum[lane] = w;
    }
    __syncthreads();
    unsigned int base = inc - tot + (wid ? wsum[wid - 1] : 0u);
#pragma unroll
    for (int k = 0; k < PER; ++k) { start[threadIdx.x * PER + k] = base; cursor[threadIdx.x * PER + k] = base; base += v[k]; }
}

__global__ void sortscatter_kernel(int N, const unsigned long long* __restrict__ keys, unsigned int* __restrict__ cursor,
                                   unsigned long long* __restrict__ bkeys)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const unsigned long long key = keys[i];
    bkeys[atomicAdd(&cursor[(unsigned int)(key >> (64 - SORT_BITS))], 1u)] = key;
}

__global__ void sortrank_kernel(int N, int NP, const unsigned long long* __restrict__ bkeys,
                                const unsigned int* __restrict__ start, int* __restrict__ order)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) { if (p < NP) order[p] = p; return; }
    const unsigned long long key = bkeys[p];
    const unsigned int b = (unsigned int)(key >> (64 - SORT_BITS));
    const unsigned int s = start[b], e = (b + 1 < SORT_NB) ? start[b + 1] : (unsigned int)N;
    unsigned int rank = 0;
    for (unsigned int q = s; q < e; ++q) rank += (bkeys[q] < key) ? 1u : 0u;
    order[s + rank] = (int)(unsigned int)(key & 0xffffffffull);
}

// a1 + a2 as a kernel of their own (genga_accel; the fused step uses fused_step.cu).  A.preshift: pending
// Sun-kick with the momentum in mom[SLOT_B].
template <int CHUNK>
__global__ void __launch_bounds__(PREP_NT)
prep_kernel(PrepArgs A, Workspace w)
{
    const double sc = A.preshift / A.M_star;
    prep_tile<CHUNK>(A, w, blockIdx.x, A.preshift != 0.0, sc * w.mom[MOM_SLOT_B + 0], sc * w.mom[MOM_SLOT_B + 1],
              sc * w.mom[MOM_SLOT_B + 2]);
}

// out[0..2] = sum_j m_j v_j, out[3] = sum_j m_j (momentum.cuh: fixed-tree, last block combines).
constexpr int MOM_NT = 256;

__global__ void __launch_bounds__(MOM_NT)
momentum_kernel(int N, const double* __restrict__ m, const double* __restrict__ v, double* __restrict__ partials,
                double* __restrict__ out, unsigned int* __restrict__ ticket)
{
    double p0 = 0, p1 = 0, p2 = 0, mt = 0;
    for (int i = blockIdx.x * MOM_NT + threadIdx.x; i < N; i += gridDim.x * MOM_NT) {
        const double mi = m[i];
        p0 = fma(mi, v[3 * i + 0], p0); p1 = fma(mi, v[3 * i + 1], p1); p2 = fma(mi, v[3 * i + 2], p2);
        mt += mi;
    }
    grid_momentum(p0, p1, p2, mt, partials, out, ticket);
}

// O7 fused with the momentum of the new velocities: v_i += tau a_i; mom[SLOT_A] = sum m v.
__global__ void __launch_bounds__(MOM_NT)
velupdate_mom_kernel(int N, double tau, const double* __restrict__ a, double* __restrict__ v,
                     const double* __restrict__ m, double* __restrict__ mom, unsigned int* __restrict__ ticket)
{
    const int i = blockIdx.x * MOM_NT + threadIdx.x;
    double p0 = 0, p1 = 0, p2 = 0, mt = 0;
    if (i < N) {
        const double mi = m[i];
        const double v0 = fma(tau, a[3 * i + 0], v[3 * i + 0]);
        const double v1 = fma(tau, a[3 * i + 1], v[3 * i + 1]);
        const double v2 = fma(tau, a[3 * i + 2], v[3 * i + 2]);
        v[3 * i + 0] = v0; v[3 * i + 1] = v1; v[3 * i + 2] = v2;
        p0 = mi * v0; p1 = mi * v1; p2 = mi * v2; mt = mi;
    }
    grid_momentum(p0, p1, p2, mt, mom + MOM_PARTIALS, mom + MOM_SLOT_A, ticket);
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

void launch_sort(const Handle* h)
{
    if (h->N == 0) return;
    unsigned int* hist = h->w.sortbuf, *start = hist + SORT_NB, *cursor = start + SORT_NB;
    cudaMemsetAsync(&h->w.ctr->extent_bits, 0, sizeof(unsigned int), h->stream);
    cudaMemsetAsync(hist, 0, SORT_NB * sizeof(unsigned int), h->stream);
    const int nb = (h->N + 255) / 256;
    extent_kernel<<<nb, 256, 0, h->stream>>>(h->N, h->w.x, &h->w.ctr->extent_bits);
    sortkey_kernel<<<nb, 256, 0, h->stream>>>(h->N, h->p.M_star, h->w.x, h->w.hcbrt, h->w.red,
                                              &h->w.ctr->extent_bits, h->w.keys, hist);
    sortscan_kernel<<<1, 1024, 0, h->stream>>>(hist, start, cursor);
    sortscatter_kernel<<<nb, 256, 0, h->stream>>>(h->N, h->w.keys, cursor, h->w.bkeys);
    sortrank_kernel<<<h->NP / 256, 256, 0, h->stream>>>(h->N, h->NP, h->w.bkeys, start, h->w.order);
}

int sort_buffer_words() { return 3 * SORT_NB; }

void launch_prep(const Handle* h, const PrepArgs& a)
{
    if (h->NP == 0) return;
    if (h->chunk == CHUNK_MIN) prep_kernel<CHUNK_MIN><<<h->NP / PREP_NT, PREP_NT, 0, h->stream>>>(a, h->w);
    else                       prep_kernel<CHUNK_MAX><<<h->NP / PREP_NT, PREP_NT, 0, h->stream>>>(a, h->w);
}

static int momentum_blocks(const Handle* h)
{
    int blocks = (h->N + MOM_NT * 4 - 1) / (MOM_NT * 4);
    if (blocks < 1) blocks = 1;
    if (blocks > h->num_sms) blocks = h->num_sms;
    return blocks;
}

void launch_momentum(const Handle* h)
{
    momentum_kernel<<<momentum_blocks(h), MOM_NT, 0, h->stream>>>(h->N, h->w.m, h->w.v, h->w.mom + MOM_PARTIALS,
                                                                   h->w.red, &h->w.ctr->ticket);
}

void launch_momentum_slot_a(const Handle* h)
{
    momentum_kernel<<<momentum_blocks(h), MOM_NT, 0, h->stream>>>(h->N, h->w.m, h->w.v, h->w.mom + MOM_PARTIALS,
                                                                   h->w.mom + MOM_SLOT_A, &h->w.ctr->ticket);
}

void launch_velupdate_mom(const Handle* h, double tau)
{
    if (h->N == 0) return;
    velupdate_mom_kernel<<<(h->N + MOM_NT - 1) / MOM_NT, MOM_NT, 0, h->stream>>>(h->N, tau, h->w.a, h->w.v, h->w.m,
                                                                                 h->w.mom, &h->w.ctr->ticket);
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

void launch_copy_v_helio(const Handle* h, const double* mom, double* out)
{
    if (h->N == 0) return;
    const int n3 = 3 * h->N;
    copy_shift_kernel<<<(n3 + 255) / 256, 256, 0, h->stream>>>(h->N, 1.0 / h->p.M_star, mom, h->w.v, out);
}

}  // namespace genga
