// kick_fp32.cu -- kernel wrappers, variants and launcher of the FP32 all-pairs kick (the kernel body
// and its description are in kick32_body.cuh).
#include <algorithm>
#include "kick32_body.cuh"

namespace genga {

namespace {

using namespace k32;

template <int I, int NT, int MINB, bool ACCS, int UNR, bool SC, int CHUNK>
__global__ void __launch_bounds__(NT, MINB)
kick32_kernel(int N, int nchunk, int nib, Workspace w, unsigned int cand_cap)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    kick32_body<I, NT, ACCS, UNR, SC, CHUNK>(N, nchunk, nib, w, cand_cap, smraw);
}

// ---- variants (genga_set_tuning key 0) ---------------------------------------------------------
typedef void (*kick32_fn)(int, int, int, Workspace, unsigned int);
struct Variant32 { kick32_fn fn[2]; int nt; int bi; size_t smem[2]; bool scaled; const char* name; };   // [0]: CHUNK 64, [1]: 128

#define V32(I_, NT_, MINB_, ACCS_, UNR_, SC_) \
    { { kick32_kernel<I_, NT_, MINB_, ACCS_, UNR_, SC_, CHUNK_MIN>, kick32_kernel<I_, NT_, MINB_, ACCS_, UNR_, SC_, CHUNK_MAX> }, \
      NT_, I_ * NT_, { sizeof(Smem32<I_, NT_, ACCS_, CHUNK_MIN>), sizeof(Smem32<I_, NT_, ACCS_, CHUNK_MAX>) }, SC_, \
      "I" #I_ " NT" #NT_ " minB" #MINB_ " accS" #ACCS_ " unr" #UNR_ " scaled" #SC_ }

const Variant32 g_variants32[] = {
    V32(2, 256, 2, false, 4, false),     // 0: default.  Plain j-records (x - o, G m): robust for any mass spectrum
    V32(2, 256, 2, true, 2, false),
    V32(2, 128, 4, false, 4, false),
    V32(2, 256, 2, false, 4, true),      // 3: mass-scaled j-records, 11 instead of 12 FMA-pipe operations per pair;
    V32(2, 256, 2, true, 4, true),       //    usually the fastest for discs of comparable masses (genga_autotune picks it);
    V32(2, 128, 4, false, 4, true),      //    chunks holding massless bodies are always handed to the FP64 near field
    V32(1, 512, 1, false, 4, true),
};
constexpr int NVAR32 = (int)(sizeof(g_variants32) / sizeof(g_variants32[0]));
const Variant32& variant32(int v)
{
    return g_variants32[(v < 0 || v >= NVAR32) ? 0 : v];
}

}  // namespace

int kick32_num_variants() { return NVAR32; }
bool kick32_variant_scaled(int v) { return (v >= 0 && v < NVAR32) ? g_variants32[v].scaled : false; }
const char* kick32_variant_name(int v) { return (v >= 0 && v < NVAR32) ? g_variants32[v].name : ""; }

// Grid of the current variant: SMs x resident CTAs.  The occupancy query and the dynamic-smem opt-in
// are per device and per variant; the result is cached in the handle (one handle = one device).
int kick32_grid(const Handle* h)
{
    const int v = h->tune[0];
    Handle* hm = const_cast<Handle*>(h);
    const int ci = (h->chunk == CHUNK_MIN) ? 0 : 1;
    if (hm->grid_cache[0][0] != v + 1) {
        const Variant32& V = variant32(v);
        cudaFuncSetAttribute(V.fn[ci], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)V.smem[ci]);
        int occ = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, V.fn[ci], V.nt, V.smem[ci]);
        if (occ < 1) occ = 1;
        hm->grid_cache[0][0] = v + 1;
        hm->grid_cache[0][1] = h->num_sms * occ;
    }
    return hm->grid_cache[0][1];
}

void launch_kick32(const Handle* h)
{
    if (h->N == 0) return;
    const Variant32& V = variant32(h->tune[0]);
    const int nib = (h->N + V.bi - 1) / V.bi;          // i-blocks that hold a live body
    const long long U = (long long)nib * h->nchunk;
    // Grid: up to four waves of CTAs (the hardware hands out the later ones as SMs free up, which evens out the
    // CTAs' unequal near-field load and keeps two CTAs resident per SM to the end), but at least 16 chunks per
    // CTA; genga_set_tuning key 2 overrides it (grid in half waves).
    const long long wave = kick32_grid(h);
    long long G = std::min(4 * wave, std::max(wave, U / 16));
    if (h->tune[2] > 0) G = wave * h->tune[2] / 2;
    if (G > U) G = U;
    if (G < 1) G = 1;
    const int ci = (h->chunk == CHUNK_MIN) ? 0 : 1;
    V.fn[ci]<<<(int)G, V.nt, V.smem[ci], h->stream>>>(h->N, h->nchunk, nib, h->w, (unsigned int)h->cand_cap);
}

}  // namespace genga
