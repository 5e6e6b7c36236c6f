// mega_step.cu -- one step of a SMALL system in ONE cooperative kernel.  For N below a few thousand the
// three launches of a step (per-body kernel, all-pairs kernel, near field) cost more than their work
// (the left end of the paper's Fig. 1, is bound by kernel-call overhead as well), so the
// same three device functions run as phases of one grid, separated by grid.sync():
//   [v += tau a] [S D] [S, r_crit, pack]  |  all-pairs kick (FP32 or FP64)  |  FP64 near field + pair list.
// The arithmetic is the separate kernels' (the same device functions); the all-pairs phase uses the
// default tiling variant with plain j-records.
#include "onbody_body.cuh"
#include "kick32_body.cuh"
#include "kick64_body.cuh"
#include "nearfield_body.cuh"

namespace genga {

namespace {

namespace cg = cooperative_groups;

constexpr int MEGA_NT = 256;
static_assert(MEGA_NT == ob::FUSED_NT, "the per-body phase needs 256-thread blocks");

template <int CHUNK, int PREC>
__global__ void __launch_bounds__(MEGA_NT, 2)
step_kernel(OnBodyArgs A, nf::NfParams P, int nchunk, int nib, Workspace w, unsigned int cand_cap)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    cg::grid_group grid = cg::this_grid();
    ob::onbody_body<CHUNK>(A, w, grid);                       // ends with r_crit / packing / zeroed a / reset counters
    grid.sync();
    if (PREC == GENGA_FP32) k32::kick32_body<2, MEGA_NT, false, 4, false, CHUNK>(A.prep.N, nchunk, nib, w, cand_cap, smraw);
    else                    k64::kick64_body<2, MEGA_NT, 8, CHUNK>(A.prep.N, nchunk, nib, w, cand_cap, smraw);
    grid.sync();
    nf::nearfield_body<CHUNK, MEGA_NT / 32>(P, w);
}

template <int CHUNK, int PREC>
constexpr size_t mega_smem()
{
    return PREC == GENGA_FP32 ? sizeof(k32::Smem32<2, MEGA_NT, false, CHUNK>) : sizeof(k64::Smem64<2, MEGA_NT, CHUNK>);
}

struct MegaFn { const void* fn; size_t smem; };

MegaFn mega_fn(int chunk, int precision)
{
    if (chunk == CHUNK_MIN) {
        if (precision == GENGA_FP32) return {(const void*)step_kernel<CHUNK_MIN, GENGA_FP32>, mega_smem<CHUNK_MIN, GENGA_FP32>()};
        return {(const void*)step_kernel<CHUNK_MIN, GENGA_FP64>, mega_smem<CHUNK_MIN, GENGA_FP64>()};
    }
    if (precision == GENGA_FP32) return {(const void*)step_kernel<CHUNK_MAX, GENGA_FP32>, mega_smem<CHUNK_MAX, GENGA_FP32>()};
    return {(const void*)step_kernel<CHUNK_MAX, GENGA_FP64>, mega_smem<CHUNK_MAX, GENGA_FP64>()};
}

}  // namespace

// Co-resident blocks of the one-kernel step for this handle's chunk size and the given precision
// (also opts the kernel in to its dynamic shared memory).  0 if it cannot run.
int mega_max_blocks(const Handle* h, int precision)
{
    const MegaFn F = mega_fn(h->chunk, precision);
    if (cudaFuncSetAttribute(F.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F.smem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, F.fn, MEGA_NT, F.smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    long long b = (long long)occ * h->num_sms;
    if (b > MOM_MAX_BLOCKS) b = MOM_MAX_BLOCKS;
    return (int)b;
}

cudaError_t launch_step_mega(const Handle* h, const OnBodyArgs& a, int precision, int max_blocks)
{
    if (h->N == 0) return cudaSuccess;
    const MegaFn F = mega_fn(h->chunk, precision);
    const int BI = 2 * MEGA_NT;
    int nib = (h->N + BI - 1) / BI;
    const long long U = (long long)nib * h->nchunk;
    long long blocks = h->NP / MEGA_NT;                       // enough for the per-body phases ...
    if (U > blocks) blocks = U;                               // ... and one (i-block, chunk) unit per CTA if there are that many
    if (blocks > max_blocks) blocks = max_blocks;
    OnBodyArgs args = a;
    nf::NfParams P = nf::make_nf_params(h);
    int nchunk = h->nchunk;
    Workspace ws = h->w;
    unsigned int cand_cap = (unsigned int)h->cand_cap;
    void* params[] = {&args, &P, &nchunk, &nib, &ws, &cand_cap};
    return cudaLaunchCooperativeKernel(F.fn, dim3((unsigned int)blocks), dim3(MEGA_NT), params, F.smem, h->stream);
}

}  // namespace genga
