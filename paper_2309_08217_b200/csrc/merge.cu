// merge.cu -- NEXT-4: perfect mergers at a step end (reading R13).
//
// Bodies i, j collide iff r_ij < R_i + R_j (strict, FP64) at the positions of the last force evaluation.  The
// candidates are the pairs of the encounter list that evaluation left (r_ij < r_crit,ij; the physical radii lie
// far inside the critical radius, which merge_init_kernel checks per body).  Every connected component of the
// collision graph becomes one body at its smallest index; the arrays are closed up in order.  In TP2 mode the list
// holds only pairs with a big body (small bodies do not see each other, readings R9 + R13) and n_big follows the
// survivors among the big bodies.
//
// A rare, tiny operation (a few pairs per step): one block does it, in phases separated by __syncthreads():
//   1 labels: label[k] = smallest index reachable from k, by relabelling over the colliding pairs until stable;
//   2 every member of a component zeroes (root) / adds to (all) the root's accumulators
//     (sum m, sum m x, sum m v, sum R^3), which live in the per-evaluation arrays pk64 / aux (rebuilt by the
//     next prep step);
//   3 roots take the merged state;
//   4 stable compaction of m, x, v, R through the staging array vtmp; newidx for the caller.
#include "genga_internal.cuh"

namespace genga {
namespace {

constexpr int MERGE_THREADS = 1024;

// label[i] = i, flag[i] = 0; status bit 2 if a body's radius exceeds half its critical radius (then the encounter
// list need not contain every colliding pair).
// A body absorbed by a merger inside an encounter integration (reading R14: absorb[i] >= 0, possibly a chain) starts
// with the label of the body that took it, so that the compaction below removes it and newidx maps it there.
__global__ void merge_init_kernel(int N, const double* __restrict__ R, const double* __restrict__ rcrit,
                                  int* __restrict__ label, int* __restrict__ flag, int* __restrict__ newidx,
                                  unsigned int* __restrict__ status, const int* __restrict__ absorb)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int r = i;
    while (absorb[r] >= 0) r = absorb[r];
    label[i] = r;
    flag[i] = 0;
    if (newidx) newidx[i] = i;                 // what it stays when nothing collides (the usual step)
    if (R[i] > 0.0 && !(2.0 * R[i] <= rcrit[i])) atomicOr(status, 2u);
}

__device__ __forceinline__ bool collide(const double* __restrict__ x, const double* __restrict__ R, int i, int j)
{
    const double dx = x[3 * j] - x[3 * i], dy = x[3 * j + 1] - x[3 * i + 1], dz = x[3 * j + 2] - x[3 * i + 2];
    return sqrt(dx * dx + dy * dy + dz * dz) < R[i] + R[j];
}

__device__ void compact(int N, int width, const int* __restrict__ label, const int* __restrict__ where,
                        double* __restrict__ arr, double* __restrict__ stage, int n_new)
{
    for (int i = threadIdx.x; i < N; i += blockDim.x)
        if (label[i] == i)
            for (int d = 0; d < width; ++d) stage[(size_t)width * where[i] + d] = arr[(size_t)width * i + d];
    __syncthreads();
    for (int k = threadIdx.x; k < n_new * width; k += blockDim.x) arr[k] = stage[k];
    __syncthreads();
}

__global__ void __launch_bounds__(MERGE_THREADS)
merge_kernel(int N, unsigned int pair_cap, const int2* __restrict__ pairs, Counters* ctr,
             double* m, double* x, double* v, double* R,
             int* label, int* flag, double4* acc1, double4* acc2,
             double* stage, int* newidx, int n_big, unsigned int* out /* [0] N', [1] status, [2] n_big' */)
{
    __shared__ int s_changed, s_any, s_nbig;
    __shared__ int s_scan[MERGE_THREADS];
    const int t = threadIdx.x;
    unsigned int np = ctr->pair_count;
    if (np > pair_cap) { np = pair_cap; if (t == 0) atomicOr(&out[1], 1u); }      // list overflowed: pairs may be missing

    // 0 ---- the usual step: no listed pair overlaps, nothing to do (newidx is the identity already)
    if (t == 0) s_any = ctr->enc_merged ? 1 : 0;      // absorbed bodies wait to be removed (reading R14)
    __syncthreads();
    for (unsigned int p = t; p < np; p += MERGE_THREADS) {
        const int2 ij = pairs[p];
        if (collide(x, R, ij.x, ij.y)) s_any = 1;
    }
    __syncthreads();
    if (!s_any) { if (t == 0) { out[0] = (unsigned int)N; out[2] = (unsigned int)(n_big > 0 ? n_big : 0); } return; }

    // 1 ---- components of the collision graph
    for (;;) {
        __syncthreads();
        if (t == 0) s_changed = 0;
        __syncthreads();
        for (unsigned int p = t; p < np; p += MERGE_THREADS) {
            const int2 ij = pairs[p];
            if (!collide(x, R, ij.x, ij.y)) continue;
            const int li = ((volatile int*)label)[ij.x], lj = ((volatile int*)label)[ij.y];
            if (li != lj) {
                const int lo = li < lj ? li : lj;
                atomicMin(&label[ij.x], lo); atomicMin(&label[ij.y], lo);
                s_changed = 1;
            }
        }
        __syncthreads();
        if (!s_changed) break;
    }

    // bodies absorbed earlier follow the body that took them to its component's root
    for (int i = t; i < N; i += MERGE_THREADS) { const int l = label[i]; if (l != i) label[i] = label[l]; }
    __syncthreads();

    // 2 ---- accumulators of the roots: zero, then every member adds itself
    for (unsigned int p = t; p < np; p += MERGE_THREADS) {
        const int2 ij = pairs[p];
        if (!collide(x, R, ij.x, ij.y)) continue;
        const int root = label[ij.x];
        if (atomicCAS(&flag[root], 0, 1) == 0) {
            acc1[root] = make_double4(0.0, 0.0, 0.0, 0.0);
            acc2[root] = make_double4(0.0, 0.0, 0.0, 0.0);
        }
    }
    __syncthreads();
    for (unsigned int p = t; p < np; p += MERGE_THREADS) {
        const int2 ij = pairs[p];
        if (!collide(x, R, ij.x, ij.y)) continue;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int k = e ? ij.y : ij.x;
            const int root = label[k];
            const int claimed = (k == root) ? atomicCAS(&flag[k], 1, 3) == 1 : atomicCAS(&flag[k], 0, 2) == 0;
            if (!claimed) continue;
            const double mk = m[k], rk = R[k];
            double* a1 = reinterpret_cast<double*>(&acc1[root]);
            double* a2 = reinterpret_cast<double*>(&acc2[root]);
            atomicAdd(a1 + 0, mk);
            atomicAdd(a1 + 1, mk * x[3 * k]); atomicAdd(a1 + 2, mk * x[3 * k + 1]); atomicAdd(a1 + 3, mk * x[3 * k + 2]);
            atomicAdd(a2 + 0, rk * rk * rk);
            atomicAdd(a2 + 1, mk * v[3 * k]); atomicAdd(a2 + 2, mk * v[3 * k + 1]); atomicAdd(a2 + 3, mk * v[3 * k + 2]);
        }
    }
    __syncthreads();

    // 3 ---- roots (flag 3) take the merged state; a massless component keeps its root's x, v.  No pair is
    //        tested after this point, so x and R may change.
    for (int k = t; k < N; k += MERGE_THREADS) {
        if (flag[k] != 3) continue;
        const double4 a1 = acc1[k], a2 = acc2[k];
        if (a1.x > 0.0) {
            x[3 * k] = a1.y / a1.x; x[3 * k + 1] = a1.z / a1.x; x[3 * k + 2] = a1.w / a1.x;
            v[3 * k] = a2.y / a1.x; v[3 * k + 1] = a2.z / a1.x; v[3 * k + 2] = a2.w / a1.x;
        }
        m[k] = a1.x;
        R[k] = cbrt(a2.x);
    }
    __syncthreads();

    // 4 ---- close up the arrays in order: where[i] = number of survivors before i (kept in flag[])
    const int seg = (N + MERGE_THREADS - 1) / MERGE_THREADS;
    const int lo = min(t * seg, N), hi = min(lo + seg, N);
    int cnt = 0, cnt_big = 0;                        // TP2 mode: the survivors among the first n_big stay the big bodies
    if (t == 0) s_nbig = 0;
    __syncthreads();
    for (int i = lo; i < hi; ++i) { const int keep = (label[i] == i); cnt += keep; cnt_big += keep && i < n_big; }
    if (cnt_big) atomicAdd(&s_nbig, cnt_big);
    s_scan[t] = cnt;
    __syncthreads();
    for (int off = 1; off < MERGE_THREADS; off <<= 1) {
        const int add = t >= off ? s_scan[t - off] : 0;
        __syncthreads();
        s_scan[t] += add;
        __syncthreads();
    }
    const int n_new = s_scan[MERGE_THREADS - 1];
    int w = s_scan[t] - cnt;
    for (int i = lo; i < hi; ++i) if (label[i] == i) flag[i] = w++;
    __syncthreads();
    if (newidx) for (int i = t; i < N; i += MERGE_THREADS) newidx[i] = flag[label[i]];
    if (n_new < N) {
        compact(N, 3, label, flag, x, stage, n_new);
        compact(N, 3, label, flag, v, stage, n_new);
        compact(N, 1, label, flag, m, stage, n_new);
        compact(N, 1, label, flag, R, stage, n_new);
    }
    if (t == 0) { out[0] = (unsigned int)n_new; out[2] = (unsigned int)s_nbig; }
}

}  // namespace

void launch_merge(const Handle* h, int* newidx_dev)
{
    if (h->N == 0) return;
    int* label = h->w.glabel;
    int* flag = h->w.glabel + h->NP;
    unsigned int* out = &h->w.ctr->merge_n;
    cudaMemsetAsync(out, 0, 3 * sizeof(unsigned int), h->stream);
    merge_init_kernel<<<(h->N + 255) / 256, 256, 0, h->stream>>>(h->N, h->w.radius, h->w.rcrit, label, flag, newidx_dev, out + 1, h->w.absorb);
    merge_kernel<<<1, MERGE_THREADS, 0, h->stream>>>(h->N, (unsigned int)h->pair_cap, h->w.pairs, h->w.ctr,
                                                     h->w.m, h->w.x, h->w.v, h->w.radius, label, flag,
                                                     h->w.pk64, h->w.aux, h->w.vtmp, newidx_dev,
                                                     (h->p.n_big >= 0 && h->p.n_big < h->N) ? h->p.n_big : -1, out);
    // the bodies absorbed inside encounter integrations (reading R14) are gone now
    cudaMemsetAsync(h->w.absorb, 0xff, (size_t)h->NP * sizeof(int), h->stream);
    cudaMemsetAsync(&h->w.ctr->enc_merged, 0, sizeof(unsigned int), h->stream);
}

}  // namespace genga
