// nearfield.cu -- kernel wrappers and launchers of the FP64 near-field pass (body and description in
// nearfield_body.cuh) and the TP2-mode kernel.
#include "nearfield_body.cuh"

namespace genga {

namespace {

using namespace nf;

template <int CHUNK>
__global__ void __launch_bounds__(128, 8)
nearfield_kernel(NfParams P, Workspace w)
{
    nearfield_body<CHUNK, 128 / 32>(P, w);
}

// ---- TP2 mode (reading R9) -----------------------------------------------------
// Only pairs with at least one big body (body index < n_big) interact, so the force evaluation
// is O(n_big N): one block row per big body b, each thread takes a few j-slots.  Per pair, in
// FP64: the force of j on b (block-reduced, one atomicAdd per block) and, unless j is big itself
// (then its own row does it), the reaction of b on j (one atomicAdd per j and big body); the
// exact r < r_crit test feeds the encounter list (big-big pairs once, from the lower index).
constexpr int TP2_NT = 128;
constexpr int TP2_JPT = 4;                         // j-slots per thread

__global__ void __launch_bounds__(TP2_NT)
tp2_kernel(NfParams P, int n_big, Workspace w)
{
    __shared__ double sred[TP2_NT / 32][3];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int b = blockIdx.y; b < n_big; b += gridDim.y) {
        const IBody I = load_ibody(w, w.bigslot[b]);          // I.body == b
        const double gmb = w.pk64[I.slot].w;
        double fx = 0.0, fy = 0.0, fz = 0.0;
#pragma unroll
        for (int t = 0; t < TP2_JPT; ++t) {
            const int sj = (blockIdx.x * TP2_JPT + t) * TP2_NT + threadIdx.x;
            bool enc = false;
            int bj = 0;
            if (sj < P.N && sj != I.slot) {
                const double4 q = w.pk64[sj];
                const double4 A = w.aux[sj];
                bj = w.order[sj];
                const double dx = q.x - I.x, dy = q.y - I.y, dz = q.z - I.z;
                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                const double r  = sqrt(r2);
                const double rc = pair_rcrit(P, I.m, A.x, I.rc, A.y, I.a, A.z, I.vk, A.w);
                const bool jbig = bj < n_big;
                enc = (r < rc) && (!jbig || I.body < bj);      // coincident bodies (r = 0) are an encounter
                if (r > 0.0) {
                    const double W = changeover(r, rc, P.weight_mode);
                    if (W != 0.0) {
                        const double u = W / (r2 * r);
                        const double sb = q.w * u;               // on b from j
                        fx = fma(sb, dx, fx); fy = fma(sb, dy, fy); fz = fma(sb, dz, fz);
                        if (!jbig) {                             // on j from b
                            const double sjb = -gmb * u;
                            atomicAdd(&w.a[3 * bj + 0], sjb * dx);
                            atomicAdd(&w.a[3 * bj + 1], sjb * dy);
                            atomicAdd(&w.a[3 * bj + 2], sjb * dz);
                        }
                    }
                }
            }
            append_pair(enc, min(I.body, bj), max(I.body, bj), w, P.pair_cap);
        }
        fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
        __syncthreads();
        if (lane == 0) { sred[wid][0] = fx; sred[wid][1] = fy; sred[wid][2] = fz; }
        __syncthreads();
        if (threadIdx.x == 0) {
            double t0 = 0, t1 = 0, t2 = 0;
            for (int k = 0; k < TP2_NT / 32; ++k) { t0 += sred[k][0]; t1 += sred[k][1]; t2 += sred[k][2]; }
            atomicAdd(&w.a[3 * I.body + 0], t0);
            atomicAdd(&w.a[3 * I.body + 1], t1);
            atomicAdd(&w.a[3 * I.body + 2], t2);
        }
    }
}

}  // namespace

void launch_nearfield(const Handle* h)
{
    if (h->N == 0) return;
    NfParams P = make_nf_params(h);
    P.gather = 1;
    int blocks = h->num_sms * 16;
    const long long need = ((long long)h->N + 15) / 16;          // a warp per four bodies is plenty (candidates << N)
    if (blocks > need && need > 0) blocks = (int)((need < h->num_sms) ? h->num_sms : need);
    if (h->chunk == CHUNK_MIN) nearfield_kernel<CHUNK_MIN><<<blocks, 128, 0, h->stream>>>(P, h->w);
    else                       nearfield_kernel<CHUNK_MAX><<<blocks, 128, 0, h->stream>>>(P, h->w);
}

void launch_tp2(const Handle* h)
{
    if (h->N == 0 || h->p.n_big <= 0) return;
    const NfParams P = make_nf_params(h);
    const int per_block = TP2_NT * TP2_JPT;
    dim3 grid((h->N + per_block - 1) / per_block, h->p.n_big < 65535 ? h->p.n_big : 65535);
    tp2_kernel<<<grid, TP2_NT, 0, h->stream>>>(P, h->p.n_big, h->w);
}

}  // namespace genga
