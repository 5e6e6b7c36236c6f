// kick_fp64.cu -- kernel wrappers, variants and launcher of the FP64 all-pairs kick (the kernel body
// and its description are in kick64_body.cuh).
#include <algorithm>
#include "kick64_body.cuh"

namespace genga {

namespace {

using namespace k64;

template <int I, int NT, int MINB, int UNR, int CHUNK>
__global__ void __launch_bounds__(NT, MINB)
kick64_kernel(int N, int nchunk, int nib, Workspace w, unsigned int cand_cap)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    kick64_body<I, NT, UNR, CHUNK>(N, nchunk, nib, w, cand_cap, smraw);
}

typedef void (*kick64_fn)(int, int, int, Workspace, unsigned int);
struct Variant64 { kick64_fn fn[2]; int nt; int bi; size_t smem[2]; const char* name; };   // [0]: CHUNK 64, [1]: 128

#define V64(I_, NT_, MINB_, UNR_) \
    { { kick64_kernel<I_, NT_, MINB_, UNR_, CHUNK_MIN>, kick64_kernel<I_, NT_, MINB_, UNR_, CHUNK_MAX> }, NT_, I_ * NT_, \
      { sizeof(Smem64<I_, NT_, CHUNK_MIN>), sizeof(Smem64<I_, NT_, CHUNK_MAX>) }, "I" #I_ " NT" #NT_ " minB" #MINB_ " unr" #UNR_ }

const Variant64 g_variants64[] = {
    V64(2, 256, 2, 8),            // 0: default
    V64(2, 256, 2, 4),
    V64(2, 256, 1, 4),
    V64(2, 128, 3, 4),
    V64(1, 256, 3, 8),
};
constexpr int NVAR64 = (int)(sizeof(g_variants64) / sizeof(g_variants64[0]));
const Variant64& variant64(int v)
{
    return g_variants64[(v < 0 || v >= NVAR64) ? 0 : v];
}

}  // namespace

int kick64_num_variants() { return NVAR64; }
const char* kick64_variant_name(int v) { return (v >= 0 && v < NVAR64) ? g_variants64[v].name : ""; }

// Grid of the current variant: SMs x resident CTAs.  The occupancy query and the dynamic-smem opt-in
// are per device and per variant; the result is cached in the handle (one handle = one device).
int kick64_grid(const Handle* h)
{
    const int v = h->tune[1];
    Handle* hm = const_cast<Handle*>(h);
    const int ci = (h->chunk == CHUNK_MIN) ? 0 : 1;
    if (hm->grid_cache[1][0] != v + 1) {
        const Variant64& V = variant64(v);
        cudaFuncSetAttribute(V.fn[ci], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)V.smem[ci]);
        int occ = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, V.fn[ci], V.nt, V.smem[ci]);
        if (occ < 1) occ = 1;
        hm->grid_cache[1][0] = v + 1;
        hm->grid_cache[1][1] = h->num_sms * occ;
    }
    return hm->grid_cache[1][1];
}

void launch_kick64(const Handle* h)
{
    if (h->N == 0) return;
    const Variant64& V = variant64(h->tune[1]);
    const int nib = (h->N + V.bi - 1) / V.bi;          // i-blocks that hold a live body
    const long long U = (long long)nib * h->nchunk;
    // Grid: up to four waves of CTAs (the hardware hands out the later ones as SMs free up, which evens out the
    // CTAs' unequal near-field load and keeps two CTAs resident per SM to the end), but at least 16 chunks per
    // CTA; genga_set_tuning key 3 overrides it (grid in half waves).
    const long long wave = kick64_grid(h);
    long long G = std::min(4 * wave, std::max(wave, U / 16));
    if (h->tune[3] > 0) G = wave * h->tune[3] / 2;
    if (G > U) G = U;
    if (G < 1) G = 1;
    const int ci = (h->chunk == CHUNK_MIN) ? 0 : 1;
    V.fn[ci]<<<(int)G, V.nt, V.smem[ci], h->stream>>>(h->N, h->nchunk, nib, h->w, (unsigned int)h->cand_cap);
}

}  // namespace genga
