// fused_step.cu -- kernel wrapper and launcher of the cooperative per-body kernel of the step (body and
// description in onbody_body.cuh).
#include "onbody_body.cuh"

namespace genga {

namespace {

using namespace ob;

template <int CHUNK>
__global__ void __launch_bounds__(FUSED_NT)
onbody_kernel(OnBodyArgs A, Workspace w)
{
    cg::grid_group grid = cg::this_grid();
    onbody_body<CHUNK>(A, w, grid);
}

}  // namespace

int onbody_max_blocks(const Handle* h)
{
    int occ = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, onbody_kernel<CHUNK_MAX>, FUSED_NT, 0);
    int occ2 = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, onbody_kernel<CHUNK_MIN>, FUSED_NT, 0);
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
    if (blocks > max_blocks) blocks = max_blocks;
    OnBodyArgs args = a;
    Workspace ws = h->w;
    void* params[] = {&args, &ws};
    const void* fn = (h->chunk == CHUNK_MIN) ? (const void*)onbody_kernel<CHUNK_MIN> : (const void*)onbody_kernel<CHUNK_MAX>;
    return cudaLaunchCooperativeKernel(fn, dim3(blocks), dim3(FUSED_NT), params, 0, h->stream);
}

}  // namespace genga
