// prep_tile.cuh -- rows a1 + a2 of the path for one tile of 256 slots: critical radius (PAPER.md:49-53,
// Eq. 1), packing of the j-side arrays in the internal order, chunk frames and the conservative
// near-field bound parameters (DESIGN.md sections 3 and 6).  Shared by prep_kernel and the fused
// per-body kernel of the step (fused_step.cu).
#pragma once

#include "genga_internal.cuh"

namespace genga {

constexpr int PREP_NT = 256;

__device__ __forceinline__ unsigned int warp_max_u32(unsigned int v)
{
    return __reduce_max_sync(0xffffffffu, v);
}

// One thread per (padded) body.  Eq. 1:  r_crit,i = max(n1 R_H,i, n2 dt v_i), R_H,i = a_i (m_i/3M)^(1/3);
// a_i from vis-viva with the stored velocity (readings G2b, G2c); v_i = sqrt(G M / a_i).
// tile: which run of PREP_NT slots this block handles; (shx, shy, shz): a pending Sun-kick displacement
// (O8) added to the positions first (and written back) if do_shift.  Must be called by all PREP_NT
// threads of the block; ends with a __syncthreads, so it can be called in a loop.
template <int CHUNK>
__device__ __forceinline__ void prep_tile(const PrepArgs& A, Workspace& w, int tile, bool do_shift,
                                          double shx, double shy, double shz)
{
    __shared__ unsigned int smax[PREP_NT / 32][5];
    __shared__ float sbox[PREP_NT / 32][6];                // per warp: min and max of the live positions
    __shared__ double sgm[PREP_NT / 32];                   // per warp: G m of its first slot, and whether all 32 slots are
    __shared__ int suni[PREP_NT / 32];                     //           live with bitwise that same G m
    const int s = tile * PREP_NT + threadIdx.x;            // slot; tiles cover NP exactly (NP % 512 == 0)
    const bool live = s < A.N;
    const int i = w.order[s];                              // body held by this slot (= s for padding)

    double px = PAD_POS, py = 0.0, pz = 0.0, gm = 0.0;
    float hq = 0.f, aq = 0.f, rf = 0.f;
    double4 ax4 = make_double4(0.0, 0.0, 0.0, 0.0);
    if (live) {
        const double mu = A.G * A.M_star;
        px = w.x[3 * i + 0]; py = w.x[3 * i + 1]; pz = w.x[3 * i + 2];
        if (do_shift) {                                    // pending Sun-kick S(tau) of the fused step (O8)
            px += shx; py += shy; pz += shz;
            w.x[3 * i + 0] = px; w.x[3 * i + 1] = py; w.x[3 * i + 2] = pz;
        }
        const double vx = w.v[3 * i + 0], vy = w.v[3 * i + 1], vz = w.v[3 * i + 2];
        const double r  = sqrt(px * px + py * py + pz * pz);
        const double v2 = vx * vx + vy * vy + vz * vz;
        double sa = 1.0 / (2.0 / r - v2 / mu);
        if (!(sa > 0.0) || !isfinite(sa)) sa = r;
        const double h  = w.hcbrt[i];
        const double vk = sqrt(mu / sa);
        const double rc = fmax(A.n1 * (sa * h), A.n2 * A.dt_rcrit * vk);
        w.rcrit[i] = rc; w.semi[i] = sa; w.vkep[i] = vk;
        const double mi = w.m[i];
        gm = A.G * mi;
        ax4 = make_double4(mi, rc, sa, vk);
        if (i < A.n_big) w.bigslot[i] = s;                 // TP2 mode: where the big bodies sit

        const double lam = (double)A.lambda * (1.0 + 1.0e-6);
        double dhq, daq, drf;
        if (A.pair_rule == GENGA_PAIR_MUTUAL_HILL) {
            dhq = lam * A.n1 * 1.2599210498948732 * h;     // cbrt(2) * h_i bounds cbrt((m_i+m_j)/3M)
            daq = sa;
            drf = lam * A.n2 * A.dt_rcrit * vk;
        } else {
            dhq = lam * rc;
            daq = 1.0;
            drf = 0.0;
        }
        hq = __double2float_ru(dhq); aq = __double2float_ru(daq); rf = __double2float_ru(drf);
        if (!(hq >= 0.f)) hq = 3.0e38f;                     // NaN state: flag everything
        if (!(aq >= 0.f)) aq = 3.0e38f;
        if (!(rf >= 0.f)) rf = 3.0e38f;
    }
    w.a[3 * i + 0] = 0.0; w.a[3 * i + 1] = 0.0; w.a[3 * i + 2] = 0.0;
    w.aslot[s] = 0.0; w.aslot[A.NP + s] = 0.0; w.aslot[2 * A.NP + s] = 0.0;   // any one-to-one slot mapping zeroes it all
    w.pk64[s] = make_double4(px, py, pz, gm);
    w.aux[s]  = ax4;
    // local frame of this slot's chunk (FP32 policy P32): origin = centre of the bounding box of the chunk's live
    // bodies (any FP64 point would do; the centre halves the chunk radius against a corner), found by warp
    // reductions handed over through shared memory (a chunk is CHUNK / 32 warps of this block)
    {
        float lo0 = live ? (float)px : 3.0e38f, lo1 = live ? (float)py : 3.0e38f, lo2 = live ? (float)pz : 3.0e38f;
        float hi0 = live ? (float)px : -3.0e38f, hi1 = live ? (float)py : -3.0e38f, hi2 = live ? (float)pz : -3.0e38f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo0 = fminf(lo0, __shfl_xor_sync(0xffffffffu, lo0, o)); hi0 = fmaxf(hi0, __shfl_xor_sync(0xffffffffu, hi0, o));
            lo1 = fminf(lo1, __shfl_xor_sync(0xffffffffu, lo1, o)); hi1 = fmaxf(hi1, __shfl_xor_sync(0xffffffffu, hi1, o));
            lo2 = fminf(lo2, __shfl_xor_sync(0xffffffffu, lo2, o)); hi2 = fmaxf(hi2, __shfl_xor_sync(0xffffffffu, hi2, o));
        }
        if ((threadIdx.x & 31) == 0) {
            float* b = sbox[threadIdx.x >> 5];
            b[0] = lo0; b[1] = lo1; b[2] = lo2; b[3] = hi0; b[4] = hi1; b[5] = hi2;
        }
    }
    __syncthreads();
    auto chunk_origin = [&](int c, double& ox_, double& oy_, double& oz_) {
        float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
        for (int ww = 0; ww < CHUNK / 32; ++ww)
            for (int t = 0; t < 3; ++t) {
                lo[t] = fminf(lo[t], sbox[c * (CHUNK / 32) + ww][t]);
                hi[t] = fmaxf(hi[t], sbox[c * (CHUNK / 32) + ww][3 + t]);
            }
        const bool any = lo[0] <= hi[0] && lo[1] <= hi[1] && lo[2] <= hi[2];      // false: no live body (or NaN state)
        ox_ = any ? (double)(0.5f * lo[0] + 0.5f * hi[0]) : 0.0;
        oy_ = any ? (double)(0.5f * lo[1] + 0.5f * hi[1]) : 0.0;
        oz_ = any ? (double)(0.5f * lo[2] + 0.5f * hi[2]) : 0.0;
    };
    double ox, oy, oz;
    chunk_origin(threadIdx.x / CHUNK, ox, oy, oz);
    const double qx = px - ox, qy = py - oy, qz = pz - oz;
    float rad = 0.f;                                        // |x - o|, rounded up; padding does not count
    if (live) {
        rad = __double2float_ru(sqrt(qx * qx + qy * qy + qz * qz) * (1.0 + 1.0e-9));
        if (!(rad >= 0.f)) rad = 3.0e38f;
    }
    // FP32 j-record.  Plain form: (x - o, G m).  Mass-scaled form (A.scaled): (q (x - o), q) with
    // q = (G m)^(-1/2), so that D = q (x_j - x_i) gives G m d / r^3 = D / |D|^3 without a multiply by
    // G m.  Bodies without (usable) mass and padding get a far-away dummy (1e18, 0, 0 | 0): their
    // term underflows to exactly 0; a chunk holding a live massless body is always flagged (below).
    const bool massive = live && (gm >= 1.0e-30) && (gm <= 1.0e30);
    float q2 = 0.f;
    {
        // two planes per chunk, two bodies per float4: [CHUNK/2] (x0, x1, y0, y1), then [CHUNK/2] (z0, z1, g0, g1)
        const int cb = s & ~(CHUNK - 1), u = (s & (CHUNK - 1)) >> 1;
        float* fa = reinterpret_cast<float*>(w.pk32 + cb + u) + (s & 1);
        float* fb = reinterpret_cast<float*>(w.pk32 + cb + CHUNK / 2 + u) + (s & 1);
        if (!A.scaled) {
            fa[0] = (float)qx; fa[2] = (float)qy; fb[0] = (float)qz; fb[2] = (float)gm;
        } else if (massive) {
            const double q = rsqrt(gm);
            fa[0] = (float)(q * qx); fa[2] = (float)(q * qy); fb[0] = (float)(q * qz); fb[2] = (float)q;
            q2 = __double2float_ru(q * q * (1.0 + 1.0e-6));
        } else {
            fa[0] = 1.0e18f; fa[2] = 0.f; fb[0] = 0.f; fb[2] = 0.f;
        }
    }
    const float rfc = (A.scaled && live && !massive) ? 3.0e38f : rf;   // massless j: (i, this chunk) always FP64
    BoundP b; b.hq = hq; b.aq = aq; b.rf = rf; b.pad = live ? 1.f : 0.f;
    w.bi[s] = b;

    // per-chunk maxima (a chunk is CHUNK / 32 warps of this block); non-negative floats order like unsigned ints
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned int m0 = warp_max_u32(__float_as_uint(hq));
    unsigned int m1 = warp_max_u32(__float_as_uint(aq));
    unsigned int m2 = warp_max_u32(__float_as_uint(rfc));
    unsigned int m3 = warp_max_u32(__float_as_uint(rad));
    unsigned int m4 = warp_max_u32(__float_as_uint(q2));
    const double gm0 = __shfl_sync(0xffffffffu, gm, 0);
    const int uniw = __all_sync(0xffffffffu, live && gm == gm0);
    if (lane == 0) { smax[wid][0] = m0; smax[wid][1] = m1; smax[wid][2] = m2; smax[wid][3] = m3; smax[wid][4] = m4; sgm[wid] = gm0; suni[wid] = uniw; }
    __syncthreads();
    if (threadIdx.x < PREP_NT / CHUNK) {
        const int c = threadIdx.x;
        ChunkP q;
        unsigned int mx[5] = {0u, 0u, 0u, 0u, 0u};
        for (int ww = 0; ww < CHUNK / 32; ++ww)
            for (int t = 0; t < 5; ++t) mx[t] = max(mx[t], smax[c * (CHUNK / 32) + ww][t]);
        q.hq  = __uint_as_float(mx[0]);
        q.aq  = __uint_as_float(mx[1]);
        q.rad = __uint_as_float(mx[3]);
        // frame guard: pairs closer than floor * 2 R_chunk go to FP64 (relative rounding error of
        // the FP32 separation <= 2^-24 (1 + 2 R_chunk / r))
        q.rf  = fmaxf(__uint_as_float(mx[2]), __fmul_ru(__fmul_ru(2.0f * A.floor_rel, q.rad), 1.000001f));
        q.q2max = A.scaled ? __uint_as_float(mx[4]) : 1.0f;   // scales the bound to the kernel's r'^2 = q^2 r^2
        bool uni = true;                                    // uniform-mass chunk: the symmetric kernels then factor G m out of the pair loop
        for (int ww = 0; ww < CHUNK / 32; ++ww)
            uni = uni && suni[c * (CHUNK / 32) + ww] && sgm[c * (CHUNK / 32) + ww] == sgm[c * (CHUNK / 32)];
        q.uni = uni ? 1.f : 0.f;
        chunk_origin(c, q.ox, q.oy, q.oz);
        w.bc[tile * (PREP_NT / CHUNK) + c] = q;
    }
    if (s == 0) { w.ctr->cand_count = 0u; w.ctr->pair_count = 0u; w.ctr->overflow = 0u; }
    __syncthreads();                                       // smax / sbox may be reused by the next tile
}

}  // namespace genga
