// kick_fp64.cu -- kernel wrappers, variants and launcher of the FP64 all-pairs kick (the kernel body
// and its description are in kick64_body.cuh).
#include <algorithm>
#include "kick64_body.cuh"
#include "kick_sym_body.cuh"

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

// The symmetric kernel (kick_sym_body.cuh): every unordered pair once, independent warps (third argument: NP).
template <int CHUNK, int NW, int MINB>
__global__ void __launch_bounds__(32 * NW, MINB)
kick64_sym_kernel(int N, int nchunk, int NP, Workspace w, unsigned int cand_cap)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    ksym::kick_sym_body<false, CHUNK>(N, NP, nchunk, w, cand_cap, smraw);
}

typedef void (*kick64_fn)(int, int, int, Workspace, unsigned int);
struct Variant64 { kick64_fn fn[2]; int nt; int bi; size_t smem[2]; const char* name; int sym_nw; };   // [0]: CHUNK 64, [1]: 128; sym_nw > 0: symmetric kernel

#define V64(I_, NT_, MINB_, UNR_) \
    { { kick64_kernel<I_, NT_, MINB_, UNR_, CHUNK_MIN>, kick64_kernel<I_, NT_, MINB_, UNR_, CHUNK_MAX> }, NT_, I_ * NT_, \
      { sizeof(Smem64<I_, NT_, CHUNK_MIN>), sizeof(Smem64<I_, NT_, CHUNK_MAX>) }, "I" #I_ " NT" #NT_ " minB" #MINB_ " unr" #UNR_, 0 }
#define V64SYM(NW_, MINB_) \
    { { kick64_sym_kernel<CHUNK_MIN, NW_, MINB_>, kick64_sym_kernel<CHUNK_MAX, NW_, MINB_> }, 32 * NW_, 32 * NW_, \
      { NW_ * sizeof(ksym::WarpSm<false, CHUNK_MIN>), NW_ * sizeof(ksym::WarpSm<false, CHUNK_MAX>) }, \
      "sym NW" #NW_ " minB" #MINB_, NW_ }

const Variant64 g_variants64[] = {
    V64(2, 256, 2, 8),            // 0: default
    V64(2, 256, 2, 4),
    V64(2, 256, 1, 4),
    V64(2, 128, 3, 4),
    V64(1, 256, 3, 8),
    V64SYM(8, 2),                 // 5: every unordered pair once (Newton's third law), register ring
    V64SYM(4, 4),
    V64SYM(16, 1),
    V64SYM(12, 1),
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
    const int ci = (h->chunk == CHUNK_MIN) ? 0 : 1;
    if (V.sym_nw > 0) {                                // symmetric kernel: see launch_kick32
        const long long NTILE = (long long)h->nchunk * (h->nchunk + 1) / 2;
        const long long wave = kick64_grid(h);
        long long G = (h->tune[3] > 0) ? wave * h->tune[3] / 2 : wave;
        if (G * V.sym_nw > NTILE) G = (NTILE + V.sym_nw - 1) / V.sym_nw;
        if (G < 1) G = 1;
        V.fn[ci]<<<(int)G, V.nt, V.smem[ci], h->stream>>>(h->N, h->nchunk, h->NP, h->w, (unsigned int)h->cand_cap);
        return;
    }
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
    V.fn[ci]<<<(int)G, V.nt, V.smem[ci], h->stream>>>(h->N, h->nchunk, nib, h->w, (unsigned int)h->cand_cap);
}

}  // namespace genga
