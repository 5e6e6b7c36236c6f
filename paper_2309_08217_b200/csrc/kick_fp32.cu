// kick_fp32.cu -- kernel wrappers, variants and launcher of the FP32 all-pairs kick (the kernel body
// and its description are in kick32_body.cuh).
#include <algorithm>
#include "kick32_body.cuh"
#include "kick_sym_body.cuh"

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

// The symmetric kernel (kick_sym_body.cuh): every unordered pair once, independent warps.  Same argument list as
// the row kernel (the third argument is NP here) so that both sit in one variant table.
template <int CHUNK, int NW, int MINB>
__global__ void __launch_bounds__(32 * NW, MINB)
kick32_sym_kernel(int N, int nchunk, int NP, Workspace w, unsigned int cand_cap)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    ksym::kick_sym_body<true, CHUNK>(N, NP, nchunk, w, cand_cap, smraw);
}

// ---- variants (genga_set_tuning key 0) ---------------------------------------------------------
typedef void (*kick32_fn)(int, int, int, Workspace, unsigned int);
struct Variant32 { kick32_fn fn[2]; int nt; int bi; size_t smem[2]; bool scaled; const char* name; int sym_nw; };   // [0]: CHUNK 64, [1]: 128; sym_nw > 0: symmetric kernel

#define V32(I_, NT_, MINB_, ACCS_, UNR_, SC_) \
    { { kick32_kernel<I_, NT_, MINB_, ACCS_, UNR_, SC_, CHUNK_MIN>, kick32_kernel<I_, NT_, MINB_, ACCS_, UNR_, SC_, CHUNK_MAX> }, \
      NT_, I_ * NT_, { sizeof(Smem32<I_, NT_, ACCS_, CHUNK_MIN>), sizeof(Smem32<I_, NT_, ACCS_, CHUNK_MAX>) }, SC_, \
      "I" #I_ " NT" #NT_ " minB" #MINB_ " accS" #ACCS_ " unr" #UNR_ " scaled" #SC_, 0 }
#define V32SYM(NW_, MINB_) \
    { { kick32_sym_kernel<CHUNK_MIN, NW_, MINB_>, kick32_sym_kernel<CHUNK_MAX, NW_, MINB_> }, 32 * NW_, 32 * NW_, \
      { NW_ * sizeof(ksym::WarpSm<true, CHUNK_MIN>), NW_ * sizeof(ksym::WarpSm<true, CHUNK_MAX>) }, false, \
      "sym NW" #NW_ " minB" #MINB_ " scaledfalse", NW_ }

const Variant32 g_variants32[] = {
    V32(2, 256, 2, false, 4, false),     // 0: default.  Plain j-records (x - o, G m): robust for any mass spectrum
    V32(2, 256, 2, true, 2, false),
    V32(2, 128, 4, false, 4, false),
    V32(2, 256, 2, false, 4, true),      // 3: mass-scaled j-records, 11 instead of 12 FMA-pipe operations per pair;
    V32(2, 256, 2, true, 4, true),       //    usually the fastest for discs of comparable masses (genga_autotune picks it);
    V32(2, 128, 4, false, 4, true),      //    chunks holding massless bodies are always handed to the FP64 near field
    V32(1, 512, 1, false, 4, true),
    V32SYM(8, 2),                        // 7: every unordered pair once (Newton's third law), register ring
    V32SYM(4, 4),
    V32SYM(16, 1),
    V32SYM(12, 1),
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
    const int ci = (h->chunk == CHUNK_MIN) ? 0 : 1;
    if (V.sym_nw > 0) {
        // symmetric kernel: the tiles (A, B >= A) are cut evenly over all warps of one wave of CTAs
        // (genga_set_tuning key 2: half waves)
        const long long NTILE = (long long)h->nchunk * (h->nchunk + 1) / 2;
        const long long wave = kick32_grid(h);
        long long G = (h->tune[2] > 0) ? wave * h->tune[2] / 2 : wave;
        if (G * V.sym_nw > NTILE) G = (NTILE + V.sym_nw - 1) / V.sym_nw;
        if (G < 1) G = 1;
        V.fn[ci]<<<(int)G, V.nt, V.smem[ci], h->stream>>>(h->N, h->nchunk, h->NP, h->w, (unsigned int)h->cand_cap);
        return;
    }
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
    V.fn[ci]<<<(int)G, V.nt, V.smem[ci], h->stream>>>(h->N, h->nchunk, nib, h->w, (unsigned int)h->cand_cap);
}

}  // namespace genga
