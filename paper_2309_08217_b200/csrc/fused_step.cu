// fused_step.cu -- kernel wrapper and launcher of the cooperative per-body kernel of the step (body and
// description in onbody_body.cuh).
#include <algorithm>
#include "onbody_body.cuh"

namespace genga {

namespace {

using namespace ob;

template <int CHUNK, int ENC>
__global__ void __launch_bounds__(FUSED_NT, ENC ? 1 : 2)
onbody_kernel(OnBodyArgs A, Workspace w)
{
    cg::grid_group grid = cg::this_grid();
    onbody_body<CHUNK, ENC>(A, w, grid);
}

// Encounter groups (NEXT-1): connected components of the encounter-pair graph by label propagation over the
// pair list; glabel[b] = smallest body index of b's component, -1 for bodies in no pair (preset by the
// launcher), -2 for the bodies of a component with more than enc::GBIG members (status bit 2; they drift on
// their Kepler orbits).  Then every component gets a group index g, a slice of the member array
// (ginfo[2 g] = offset, ginfo[2 g + 1] = count) and registers its members there (in no particular order: the
// integrating team sorts them).  One block.
__global__ void __launch_bounds__(1024)
group_kernel(int NP, const int2* __restrict__ pairs, Counters* __restrict__ ctr, unsigned int pair_cap,
             int* __restrict__ glabel, int* __restrict__ ginfo, int* __restrict__ ulist, int maxgroups)
{
    __shared__ int changed;
    __shared__ int cursor;
    int* members = ginfo + 2 * (size_t)maxgroups;
    int* gcount = glabel + NP;
    const unsigned int total = ctr->pair_count;
    const unsigned int n = total < pair_cap ? total : pair_cap;
    if (threadIdx.x == 0) {
        if (total > pair_cap) atomicOr(&ctr->enc_status, 1u);               // list overflowed: groups incomplete
        ctr->enc_groups = 0u; ctr->enc_bodies = 0u; ctr->enc_maxsize = 0u;
        ctr->enc_rhs_sum = 0u; ctr->enc_rhs_max = 0u; ctr->enc_rejected = 0u;
    }
    if (n == 0) return;
    // the bodies that occur in a pair, each once (gcount is preset to -1 like the labels): every later pass
    // walks this short list instead of all N bodies
    __shared__ int nuniq;
    if (threadIdx.x == 0) { nuniq = 0; cursor = 0; }
    __syncthreads();
    for (unsigned int p = threadIdx.x; p < 2u * n; p += blockDim.x) {
        const int2 ij = pairs[p >> 1];
        const int b = (p & 1u) ? ij.y : ij.x;
        if (atomicCAS(&gcount[b], -1, 0) == -1) { glabel[b] = b; ulist[atomicAdd(&nuniq, 1)] = b; }
    }
    __syncthreads();
    const int nu = nuniq;
    for (int iter = 0; iter < (1 << 20); ++iter) {
        if (threadIdx.x == 0) changed = 0;
        __syncthreads();
        for (unsigned int p = threadIdx.x; p < n; p += blockDim.x) {
            const int2 ij = pairs[p];
            const int a = ((volatile int*)glabel)[ij.x], b = ((volatile int*)glabel)[ij.y], m = min(a, b);
            if (a != m) { atomicMin(&glabel[ij.x], m); changed = 1; }
            if (b != m) { atomicMin(&glabel[ij.y], m); changed = 1; }
        }
        __syncthreads();
        const int again = changed;
        __syncthreads();
        if (!again) break;
    }
    // member counts; components too large for the leader's arrays are dissolved (and reported)
    for (int q = threadIdx.x; q < nu; q += blockDim.x) atomicAdd(&gcount[glabel[ulist[q]]], 1);
    __syncthreads();
    for (int q = threadIdx.x; q < nu; q += blockDim.x) {
        const int b = ulist[q], l = glabel[b];
        if (l != b && gcount[l] > enc::GBIG) { glabel[b] = -2; atomicOr(&ctr->enc_status, 2u); }
    }
    __syncthreads();
    for (int q = threadIdx.x; q < nu; q += blockDim.x) { const int b = ulist[q]; if (glabel[b] == b && gcount[b] > enc::GBIG) glabel[b] = -2; }
    __syncthreads();
    for (int q = threadIdx.x; q < nu; q += blockDim.x) {
        const int b = ulist[q];
        if (glabel[b] == b) {                                               // leader of a valid group
            const unsigned int g = atomicAdd(&ctr->enc_groups, 1u);
            const int cnt = gcount[b];
            atomicAdd(&ctr->enc_bodies, (unsigned int)cnt); atomicMax(&ctr->enc_maxsize, (unsigned int)cnt);
            ginfo[2 * g] = atomicAdd(&cursor, cnt);
            ginfo[2 * g + 1] = 0;
            gcount[b] = (int)g;
        }
    }
    __syncthreads();
    for (int q = threadIdx.x; q < nu; q += blockDim.x) {
        const int b = ulist[q], l = glabel[b];
        if (l >= 0) {
            const int g = gcount[l];
            const int k = atomicAdd(&ginfo[2 * g + 1], 1);
            members[ginfo[2 * g] + k] = b;
        }
    }
}

}  // namespace

int onbody_max_blocks(const Handle* h, bool enc)
{
    int occ = 0;
    const bool full = h->p.enc_collide != 0 || h->p.enc_levels > 1;
    const void* f1 = !enc ? (const void*)onbody_kernel<CHUNK_MAX, 0> : (full ? (const void*)onbody_kernel<CHUNK_MAX, 2> : (const void*)onbody_kernel<CHUNK_MAX, 1>);
    const void* f2 = !enc ? (const void*)onbody_kernel<CHUNK_MIN, 0> : (full ? (const void*)onbody_kernel<CHUNK_MIN, 2> : (const void*)onbody_kernel<CHUNK_MIN, 1>);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, f1, FUSED_NT, 0);
    int occ2 = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, f2, FUSED_NT, 0);
    if (occ2 < occ) occ = occ2;
    if (occ < 1) occ = 1;
    long long b = (long long)occ * h->num_sms;
    if (b > MOM_MAX_BLOCKS) b = MOM_MAX_BLOCKS;
    return (int)b;
}

// Returns cudaSuccess or the launch error (cooperative launch unsupported, too large a grid, ...).
cudaError_t launch_onbody(const Handle* h, const OnBodyArgs& a, int max_blocks)
{
    if (h->N == 0) return cudaSuccess;
    int blocks = h->NP / PREP_NT;
    // with encounter groups: every co-resident CTA, whatever N -- a group takes a warp for as long as its integration lasts,
    // and a grid sized for the per-body phases (N = 10 000: 40 CTAs) made 1 100 groups queue three and four deep per warp
    if (a.enc.on && a.do_drift) blocks = max_blocks;
    if (blocks > max_blocks) blocks = max_blocks;
    OnBodyArgs args = a;
    Workspace ws = h->w;
    void* params[] = {&args, &ws};
    const void* fn;
    if (a.enc.on && a.do_drift) {
        if (a.enc.collide || a.enc.levels > 1)
            fn = (h->chunk == CHUNK_MIN) ? (const void*)onbody_kernel<CHUNK_MIN, 2> : (const void*)onbody_kernel<CHUNK_MAX, 2>;
        else
            fn = (h->chunk == CHUNK_MIN) ? (const void*)onbody_kernel<CHUNK_MIN, 1> : (const void*)onbody_kernel<CHUNK_MAX, 1>;
    } else
        fn = (h->chunk == CHUNK_MIN) ? (const void*)onbody_kernel<CHUNK_MIN, 0> : (const void*)onbody_kernel<CHUNK_MAX, 0>;
    return cudaLaunchCooperativeKernel(fn, dim3(blocks), dim3(FUSED_NT), params, 0, h->stream);
}

// Encounter groups of the pair list the last force evaluation left (encounter mode, before the drift).
cudaError_t launch_groups(const Handle* h)
{
    if (h->N == 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(h->w.glabel, 0xff, 2 * (size_t)h->NP * sizeof(int), h->stream);   // labels and counts: -1
    if (e != cudaSuccess) return e;
    group_kernel<<<1, 1024, 0, h->stream>>>(h->NP, h->w.pairs, h->w.ctr, (unsigned int)h->pair_cap, h->w.glabel, h->w.ginfo, h->w.gulist,
                                        (int)std::min((size_t)h->pair_cap, (size_t)h->NP / 2));
    return cudaGetLastError();
}

}  // namespace genga
