// kick_sym_body.cuh -- the all-pairs long-range kick with every UNORDERED pair evaluated once
// (Newton's third law), FP32 force precision or FP64.
//
//   a_i = sum_{j != i} G m_j (x_j - x_i) / r_ij^3          (pairs outside the changeover zones; the zones go to
//                                                            the FP64 near-field kernel)
// The pair (i, j) costs 3 subtractions, r^2, one MUFU seed and y^3 ONCE; the two forces G m_j y^3 d and
// -G m_i y^3 d then take 8 more operations: 16 FMA-pipe lane operations + 1 MUFU per unordered pair in FP32
// (8 + 1/2 per ordered pair, against 11-12 + 1 for the row kernel kick32_body.cuh), 20 FP64 operations in FP64
// (10 per ordered pair, against 16).
//
// Register ring.  A warp works on a TILE (chunk A, chunk B).  Lane L holds P = CHUNK/32 bodies of A
// ("stationary": positions, G m, partial sums in registers for the whole tile) and, at ring step t, faces the
// bodies of B that lane (L + t) mod 32 owns ("travelling": positions read from shared memory, their partial
// sums in registers, moved one lane on by SHFL after every step).  32 steps visit every pair of the tile
// once; after the 32nd shuffle the travelling sums are back in their owner's lane.
//
// Warps are independent.  The tiles (A, B >= A) are numbered row by row and cut evenly over all warps of the
// grid; a warp keeps the FP64 sums of its stationary chunk in its own shared memory while it stays in a row and
// copies the next travelling chunk into its own double buffer (cp.async) while it works on the current one.
// Partial sums reach memory by coalesced FP64 reductions (RED.ADD.F64, 12 per lane and tile) into aslot[], an
// accumulator in the internal order that the near-field kernel folds into a[]: the travelling sums after every
// tile, the stationary sums when the warp leaves the row.  The chunk against itself (B == A) is evaluated
// one-sidedly with the self pair masked.  No CTA-wide barrier, no inter-warp dependency.
//
// Near field (mixed-precision policy P32): a tile whose chunk spheres are farther apart
// than every bound of the two chunks holds no near pair and runs without tracking.  Otherwise the smallest
// r^2 of every (stationary body, B) and every (travelling body, A) is tracked (the travelling minima shuffle
// with their sums), and a (body, chunk) partial whose minimum is not above its bound is discarded and pushed
// to the candidate list for the FP64 near-field kernel, exactly as the row kernels do.
#pragma once

#include "tile_pipeline.cuh"

namespace genga {
namespace ksym {

typedef unsigned long long f2;   // two packed floats

__device__ __forceinline__ f2 pk(float lo, float hi)
{
    f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r;
}
__device__ __forceinline__ void upk(f2 v, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f2 add2(f2 a, f2 b)
{
    f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b)
{
    f2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r;
}
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c)
{
    f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r;
}
__device__ __forceinline__ float rsq(float a)
{
    float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r;
}
__device__ __forceinline__ double rsq64h(double a)
{
    double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r;
}
__device__ __forceinline__ float min3(float a, float b, float c)
{
    float r; asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r;
}
__device__ __forceinline__ f2 shf2(f2 v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ double shd(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }

// Shared memory of one warp.  Travelling positions: FP32 16 B per body in two planes per chunk
// ([CHUNK/2] (x0,x1,y0,y1) then [CHUNK/2] (z0,z1,Gm0,Gm1), chunk-relative), FP64 32 B per body in four planes (tile64).
template <bool F32, int CHUNK>
struct __align__(16) WarpSm {
    static constexpr int POS_BYTES = F32 ? 16 : 32;
    unsigned char pos[2][CHUNK * POS_BYTES];     // double buffer of the travelling chunk
    ChunkP   bcB[2];                             // its chunk record
    ChunkP   bcA;                                // chunk record of the stationary chunk
    double   accS[3][CHUNK];                     // FP64 sums of the stationary chunk while the warp stays in its row
    double   xiS[F32 ? 3 : 1][F32 ? CHUNK : 1];  // FP32 kernel: FP64 positions of the stationary bodies (frames)
};

__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src_gmem)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_) : "memory"); }

// aslot[]: component-major [3][NP]; inside a chunk the two bodies of pair u sit CHUNK/2 apart (body 2u + h at
// h * CHUNK/2 + u), so that the 32 lanes of a reduction hit 32 consecutive doubles.
__host__ __device__ inline int aslot_index(int slot, int chunk_size)
{
    const int b = slot & (chunk_size - 1);
    return (slot - b) + (b & 1) * (chunk_size / 2) + (b >> 1);
}

// Conservative near bound of body (hq, aq, rf) against chunk record C
__device__ __forceinline__ float bound_of(const BoundP& b, const ChunkP& C)
{
    return fmaxf(fmaxf(b.hq, C.hq) * fmaxf(b.aq, C.aq), fmaxf(b.rf, C.rf));
}

// No pair of the two chunks can be near: distance of the frame origins beyond both radii plus the largest
// bound any body of either chunk can have against the other chunk.
__device__ __forceinline__ bool tile_is_far(const ChunkP& A, const ChunkP& B)
{
    const double ex = A.ox - B.ox, ey = A.oy - B.oy, ez = A.oz - B.oz;
    const double d2 = fma(ez, ez, fma(ey, ey, ex * ex));
    const float bmax = fmaxf(fmaxf(A.hq, B.hq) * fmaxf(A.aq, B.aq), fmaxf(A.rf, B.rf));
    const double reach = ((double)bmax + (double)A.rad + (double)B.rad) * 1.00001;
    return d2 > reach * reach;
}

// ---- one tile, FP32 force precision --------------------------------------------------------------------------
// MODE 0: far tile (no tracking), 1: near tile (smallest r^2 tracked on both sides), 2: the chunk against
// itself (one-sided, self pair masked, tracking on).  Lane L owns the pairs u = L + 32 k (bodies 2u, 2u + 1)
// of a chunk, as stationary and as travelling body alike.
//   pB   set B in shared memory: planes [CHUNK/2] (x0,x1,y0,y1), [CHUNK/2] (z0,z1,Gm0,Gm1), relative to Bc's origin
//   xS   this warp's stationary FP64 positions [3][CHUNK];  gi: G m of the lane's stationary bodies
//   aS   this warp's stationary FP64 sums [3][CHUNK];  gT: aslot[] at chunk B (component stride NP)
//   UNI  (far tiles only) both chunks are uniform in mass (ChunkP::uni): G m_B and -G m_A are factored out of the pair loop
//        (14 instead of 16 packed operations per two unordered pairs) and multiplied in, in FP64, when the sums leave the tile
template <int CHUNK, int MODE, bool UNI = false>
__device__ __forceinline__ void tile32(int lane, const float4* __restrict__ pB, const ChunkP& Ac, const ChunkP& Bc,
                                       const double* __restrict__ xS, const float (&gi)[CHUNK / 32],
                                       double* __restrict__ aS, double* __restrict__ gT, int NP, int cA, int cB, int N,
                                       Workspace& w, unsigned int cand_cap)
{
    constexpr int P = CHUNK / 32, KP = CHUNK / 64;
    constexpr bool NEAR = MODE != 0, SELF = MODE == 2;
    static_assert(!UNI || MODE == 0, "mass factored out for far tiles only");
    f2 nx[P], ny[P], nz[P], ng[P], ax[P], ay[P], az[P];
    float mn[P];
    {
        const double ox = Bc.ox, oy = Bc.oy, oz = Bc.oz;       // stationary positions in B's frame: FP64 subtraction, one rounding
#pragma unroll
        for (int p = 0; p < P; ++p) {
            const int bi = 2 * (lane + 32 * (p >> 1)) + (p & 1);
            const float fx = (float)(ox - xS[0 * CHUNK + bi]);
            const float fy = (float)(oy - xS[1 * CHUNK + bi]);
            const float fz = (float)(oz - xS[2 * CHUNK + bi]);
            nx[p] = pk(fx, fx); ny[p] = pk(fy, fy); nz[p] = pk(fz, fz); ng[p] = pk(-gi[p], -gi[p]);
            ax[p] = 0ull; ay[p] = 0ull; az[p] = 0ull; mn[p] = 3.0e38f;
        }
    }
    f2 bx[KP], by[KP], bz[KP];
    float mja[KP], mjb[KP];
#pragma unroll
    for (int q = 0; q < KP; ++q) { bx[q] = 0ull; by[q] = 0ull; bz[q] = 0ull; mja[q] = 3.0e38f; mjb[q] = 3.0e38f; }
    const int src = (lane + 1) & 31;

#pragma unroll 4      // several steps per iteration: fewer register renaming moves at the loop end
    for (int st = 0; st < 32; ++st) {
        const int owner = (lane + st) & 31;
#pragma unroll
        for (int q = 0; q < KP; ++q) {
            const float4 A4 = pB[owner + 32 * q], B4 = pB[CHUNK / 2 + owner + 32 * q];
            const f2 xj = pk(A4.x, A4.y), yj = pk(A4.z, A4.w), zj = pk(B4.x, B4.y), gj = pk(B4.z, B4.w);
#pragma unroll
            for (int p = 0; p < P; ++p) {
                const f2 dx = add2(xj, nx[p]), dy = add2(yj, ny[p]), dz = add2(zj, nz[p]);
                f2 r2 = mul2(dx, dx);
                r2 = fma2(dy, dy, r2);
                r2 = fma2(dz, dz, r2);
                float r2a, r2b; upk(r2, r2a, r2b);
                float ya = rsq(r2a), yb = rsq(r2b);
                if (SELF && q == (p >> 1)) {
                    // step 0 faces the lane's own bodies: the self term is 0 by selection (d = 0 gives y = inf) and
                    // stays out of the tracking, so a chunk is flagged for itself only if a DIFFERENT body is near
                    const bool self = st == 0;
                    if (p & 1) { yb = self ? 0.f : yb; r2b = self ? 3.0e38f : r2b; }
                    else       { ya = self ? 0.f : ya; r2a = self ? 3.0e38f : r2a; }
                }
                if (NEAR) {
                    mn[p] = min3(mn[p], r2a, r2b);
                    if (!SELF) { mja[q] = fminf(mja[q], r2a); mjb[q] = fminf(mjb[q], r2b); }
                }
                const f2 y = pk(ya, yb);
                const f2 t = mul2(y, y);
                const f2 y3 = mul2(t, y);
                const f2 si = UNI ? y3 : mul2(gj, y3);         // G m_j / r^3: force on the stationary body (UNI: 1 / r^3)
                ax[p] = fma2(si, dx, ax[p]);
                ay[p] = fma2(si, dy, ay[p]);
                az[p] = fma2(si, dz, az[p]);
                if (!SELF) {
                    const f2 sj = UNI ? y3 : mul2(ng[p], y3);  // -G m_i / r^3: reaction on the travelling bodies (UNI: 1 / r^3)
                    bx[q] = fma2(sj, dx, bx[q]);
                    by[q] = fma2(sj, dy, by[q]);
                    bz[q] = fma2(sj, dz, bz[q]);
                }
            }
        }
        if (!SELF) {
#pragma unroll
            for (int q = 0; q < KP; ++q) {
                bx[q] = shf2(bx[q], src); by[q] = shf2(by[q], src); bz[q] = shf2(bz[q], src);
                if (NEAR) { mja[q] = __shfl_sync(0xffffffffu, mja[q], src); mjb[q] = __shfl_sync(0xffffffffu, mjb[q], src); }
            }
        }
    }

    // ---- tile end: keep the FP32 partials (added in FP64) or hand the (body, chunk) to the near field --------
#pragma unroll
    for (int k = 0; k < KP; ++k) {
        const int u = lane + 32 * k;
        bool keep[2] = {true, true};
        float px[2], py[2], pz[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int p = 2 * k + h;
            float lo, hi;
            upk(ax[p], lo, hi); px[h] = lo + hi;
            upk(ay[p], lo, hi); py[h] = lo + hi;
            upk(az[p], lo, hi); pz[h] = lo + hi;
            if (NEAR) {
                const int slot = cA * CHUNK + 2 * u + h;
                const float Bq = bound_of(w.bi[slot], Bc);
                keep[h] = mn[p] > ((slot < N) ? Bq * Bq : -1.0f);
                const unsigned int bal = __ballot_sync(0xffffffffu, !keep[h]);
                if (bal) push_candidates(bal, !keep[h], slot, cB, &w.ctr->cand_count, w.cand, cand_cap);
            }
        }
        double2* d;
        double2 v;
        if (UNI) {                                       // the common G m of chunk B (as the kernel sees it: the FP32 record's)
            const double gB = (double)pB[CHUNK / 2].z;
            d = reinterpret_cast<double2*>(aS + 0 * CHUNK + 2 * u); v = *d;
            v.x = fma(gB, (double)px[0], v.x); v.y = fma(gB, (double)px[1], v.y); *d = v;
            d = reinterpret_cast<double2*>(aS + 1 * CHUNK + 2 * u); v = *d;
            v.x = fma(gB, (double)py[0], v.x); v.y = fma(gB, (double)py[1], v.y); *d = v;
            d = reinterpret_cast<double2*>(aS + 2 * CHUNK + 2 * u); v = *d;
            v.x = fma(gB, (double)pz[0], v.x); v.y = fma(gB, (double)pz[1], v.y); *d = v;
            continue;
        }
        d = reinterpret_cast<double2*>(aS + 0 * CHUNK + 2 * u); v = *d;
        v.x += keep[0] ? (double)px[0] : 0.0; v.y += keep[1] ? (double)px[1] : 0.0; *d = v;
        d = reinterpret_cast<double2*>(aS + 1 * CHUNK + 2 * u); v = *d;
        v.x += keep[0] ? (double)py[0] : 0.0; v.y += keep[1] ? (double)py[1] : 0.0; *d = v;
        d = reinterpret_cast<double2*>(aS + 2 * CHUNK + 2 * u); v = *d;
        v.x += keep[0] ? (double)pz[0] : 0.0; v.y += keep[1] ? (double)pz[1] : 0.0; *d = v;
    }
    if (!SELF) {
#pragma unroll
        for (int q = 0; q < KP; ++q) {
            const int u = lane + 32 * q;
            bool keep[2] = {true, true};
            if (NEAR) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int slot = cB * CHUNK + 2 * u + h;
                    const float Bq = bound_of(w.bi[slot], Ac);
                    keep[h] = (h ? mjb[q] : mja[q]) > ((slot < N) ? Bq * Bq : -1.0f);
                    const unsigned int bal = __ballot_sync(0xffffffffu, !keep[h]);
                    if (bal) push_candidates(bal, !keep[h], slot, cA, &w.ctr->cand_count, w.cand, cand_cap);
                }
            }
            float x0, x1, y0, y1, z0, z1;
            upk(bx[q], x0, x1); upk(by[q], y0, y1); upk(bz[q], z0, z1);
            const int slot0 = cB * CHUNK + 2 * u;
            const double sc = UNI ? -(double)gi[0] : 1.0;      // UNI: the common -G m of chunk A, still to be multiplied in
            if (keep[0] && slot0 < N) {
                atomicAdd(gT + u, sc * (double)x0); atomicAdd(gT + NP + u, sc * (double)y0); atomicAdd(gT + 2 * NP + u, sc * (double)z0);
            }
            if (keep[1] && slot0 + 1 < N) {
                atomicAdd(gT + CHUNK / 2 + u, sc * (double)x1); atomicAdd(gT + NP + CHUNK / 2 + u, sc * (double)y1);
                atomicAdd(gT + 2 * NP + CHUNK / 2 + u, sc * (double)z1);
            }
        }
    }
}

// ---- one tile, FP64 ------------------------------------------------------------------------------------------
// 1/r^3 from the MUFU.RSQ64H seed y0 (|1 - r^2 y0^2| <= 2^-19.07, measured over 7.6e8 arguments) and one cubic
// correction: t = y0^2, e = 1 - r^2 t, 1/r^3 = y0^3 (1 + 3/2 e + 15/8 e^2) + O(e^3) (truncation < 1e-17).
// 20 FP64 operations per unordered pair.  The travelling set is taken two bodies per lane at a time (CHUNK/64
// rings of 32 steps), which keeps the tile in 128 registers.  Tracking compares the high words of r^2.
//   pB   set B in shared memory (absolute positions): four planes of CHUNK/2 double2, plane 2h + 0 = (x, y) and
//        plane 2h + 1 = (z, G m) of the bodies 2u + h
template <int CHUNK, int MODE, bool UNI = false>
__device__ __forceinline__ void tile64(int lane, const double2* __restrict__ pB, const ChunkP& Ac, const ChunkP& Bc,
                                       const double (&xi)[CHUNK / 32], const double (&yi)[CHUNK / 32],
                                       const double (&zi)[CHUNK / 32], const double (&gi)[CHUNK / 32],
                                       double* __restrict__ aS, double* __restrict__ gT, int NP, int cA, int cB, int N,
                                       Workspace& w, unsigned int cand_cap)
{
    constexpr int P = CHUNK / 32, KP = CHUNK / 64;
    constexpr bool NEAR = MODE != 0, SELF = MODE == 2;
    static_assert(!UNI || MODE == 0, "mass factored out for far tiles only");
    const double gB = UNI ? pB[CHUNK / 2].y : 1.0;     // UNI: the common G m of chunk B (plane 1, entry 0: body 0's (z, G m)) ...
    const double gA = UNI ? gi[0] : 1.0;               // ... and of chunk A: 18 instead of 20 FP64 operations per unordered pair
    double ax[P], ay[P], az[P];
    int mn[P];
#pragma unroll
    for (int p = 0; p < P; ++p) { ax[p] = 0.0; ay[p] = 0.0; az[p] = 0.0; mn[p] = 0x7fffffff; }
    const int src = (lane + 1) & 31;

#pragma unroll 1
    for (int k = 0; k < KP; ++k) {
        double bx[2] = {0.0, 0.0}, by[2] = {0.0, 0.0}, bz[2] = {0.0, 0.0};
        int mj[2] = {0x7fffffff, 0x7fffffff};
#pragma unroll 1
        for (int st = 0; st < 32; ++st) {
            const int u = ((lane + st) & 31) + 32 * k;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const double2 Jxy = pB[(2 * h) * (CHUNK / 2) + u], Jzg = pB[(2 * h + 1) * (CHUNK / 2) + u];
                const double4 J = make_double4(Jxy.x, Jxy.y, Jzg.x, Jzg.y);
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const double dx = J.x - xi[p], dy = J.y - yi[p], dz = J.z - zi[p];
                    double r2 = dx * dx;
                    r2 = fma(dy, dy, r2);
                    r2 = fma(dz, dz, r2);
                    double y0 = rsq64h(r2);
                    int r2h = __double2hiint(r2);
                    if (SELF && (p & 1) == h) {
                        // ring k, step 0 faces the lane's own pair: the self term is 0 by selection, untracked
                        const bool self = (st == 0) && ((p >> 1) == k);
                        y0 = self ? 0.0 : y0;
                        r2h = self ? 0x7fffffff : r2h;
                    }
                    if (NEAR) {
                        mn[p] = min(mn[p], r2h);
                        if (!SELF) mj[h] = min(mj[h], r2h);
                    }
                    const double t  = y0 * y0;
                    const double e  = fma(-r2, t, 1.0);
                    const double c  = fma(1.875, e, 1.5);
                    const double y3 = y0 * t;
                    const double ye = y3 * e;
                    const double s0 = fma(ye, c, y3);
                    const double si = UNI ? s0 : J.w * s0;
                    ax[p] = fma(si, dx, ax[p]);
                    ay[p] = fma(si, dy, ay[p]);
                    az[p] = fma(si, dz, az[p]);
                    if (!SELF) {
                        const double sj = UNI ? s0 : gi[p] * s0;
                        bx[h] = fma(-sj, dx, bx[h]);
                        by[h] = fma(-sj, dy, by[h]);
                        bz[h] = fma(-sj, dz, bz[h]);
                    }
                }
            }
            if (!SELF) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    bx[h] = shd(bx[h], src); by[h] = shd(by[h], src); bz[h] = shd(bz[h], src);
                    if (NEAR) mj[h] = __shfl_sync(0xffffffffu, mj[h], src);
                }
            }
        }
        if (!SELF) {                                   // the travelling sums of ring k are home: lane's pair u = lane + 32 k
            const int u = lane + 32 * k;
            bool keep[2] = {true, true};
            if (NEAR) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int slot = cB * CHUNK + 2 * u + h;
                    const float Bq = bound_of(w.bi[slot], Ac);
                    const double bd = (double)Bq * (double)Bq * 1.000001;      // equal high words count as near
                    keep[h] = mj[h] > ((slot < N) ? __double2hiint(bd) : -1);
                    const unsigned int bal = __ballot_sync(0xffffffffu, !keep[h]);
                    if (bal) push_candidates(bal, !keep[h], slot, cA, &w.ctr->cand_count, w.cand, cand_cap);
                }
            }
            const int slot0 = cB * CHUNK + 2 * u;
            if (keep[0] && slot0 < N) {
                atomicAdd(gT + u, gA * bx[0]); atomicAdd(gT + NP + u, gA * by[0]); atomicAdd(gT + 2 * NP + u, gA * bz[0]);
            }
            if (keep[1] && slot0 + 1 < N) {
                atomicAdd(gT + CHUNK / 2 + u, gA * bx[1]); atomicAdd(gT + NP + CHUNK / 2 + u, gA * by[1]);
                atomicAdd(gT + 2 * NP + CHUNK / 2 + u, gA * bz[1]);
            }
        }
    }

#pragma unroll
    for (int k = 0; k < KP; ++k) {
        const int u = lane + 32 * k;
        bool keep[2] = {true, true};
        if (NEAR) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int slot = cA * CHUNK + 2 * u + h;
                const float Bq = bound_of(w.bi[slot], Bc);
                const double bd = (double)Bq * (double)Bq * 1.000001;
                keep[h] = mn[2 * k + h] > ((slot < N) ? __double2hiint(bd) : -1);
                const unsigned int bal = __ballot_sync(0xffffffffu, !keep[h]);
                if (bal) push_candidates(bal, !keep[h], slot, cB, &w.ctr->cand_count, w.cand, cand_cap);
            }
        }
        double2* d;
        double2 v;
        d = reinterpret_cast<double2*>(aS + 0 * CHUNK + 2 * u); v = *d;
        v.x += keep[0] ? gB * ax[2 * k] : 0.0; v.y += keep[1] ? gB * ax[2 * k + 1] : 0.0; *d = v;
        d = reinterpret_cast<double2*>(aS + 1 * CHUNK + 2 * u); v = *d;
        v.x += keep[0] ? gB * ay[2 * k] : 0.0; v.y += keep[1] ? gB * ay[2 * k + 1] : 0.0; *d = v;
        d = reinterpret_cast<double2*>(aS + 2 * CHUNK + 2 * u); v = *d;
        v.x += keep[0] ? gB * az[2 * k] : 0.0; v.y += keep[1] ? gB * az[2 * k + 1] : 0.0; *d = v;
    }
}

// ---- the kernel as a device function -------------------------------------------------------------------------
// smraw: (blockDim.x / 32) * sizeof(WarpSm<F32, CHUNK>) bytes of 16-byte aligned shared memory.  NP: padded body
// count (component stride of aslot[]).
template <bool F32, int CHUNK>
__device__ __forceinline__ void kick_sym_body(int N, int NP, int nchunk, Workspace& w, unsigned int cand_cap, unsigned char* smraw)
{
    typedef WarpSm<F32, CHUNK> Sm;
    constexpr int P = CHUNK / 32;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    Sm& sm = reinterpret_cast<Sm*>(smraw)[wid];

    // tiles (A, B >= A), row by row: row A starts at tile A n - A (A - 1) / 2 and has n - A tiles
    const long long n = nchunk;
    const long long NTILE = n * (n + 1) / 2;
    // Which range gw of the tiles a warp takes.  (1) Neighbouring ranges go to different SMs: the ranges are not equally
    // dear -- the last ones are the short rows at the corner of the triangle, all diagonal and near tiles and a row change
    // every few tiles -- and with CTA b holding the ranges 12 b .. 12 b + 11 the last dozen SMs finished 20 % after the
    // others (N = 16 384).  (2) The warps that share a sub-partition (wid, wid + 4, ...) take ADJACENT ranges: the issue
    // slots of a sub-partition are what the ring loops compete for, and adjacent ranges differ by at most one tile in
    // all (N = 16 384: 13 or 14 tiles per sub-partition; ranges a multiple of 37 apart all had 4, or all 5: 12 or 15).
    // (2) puts three dear ranges into one sub-partition, though, where (1) alone has one dear warp among the twelve of an
    // SM: with many tiles per warp, where the counts hardly matter, (1) alone is better (N = 40 000: 0.441 against 0.458 ms).
    const int nwq = (int)(blockDim.x >> 7);                          // warps per sub-partition
    const long long nwarp = (long long)gridDim.x * (blockDim.x >> 5);
    const long long gw = (NTILE < 12 * nwarp) ? ((long long)blockIdx.x + (long long)gridDim.x * (wid & 3)) * nwq + (wid >> 2)
                                              : (long long)wid * gridDim.x + blockIdx.x;
    long long t = (NTILE * gw) / nwarp;
    const long long t1 = (NTILE * (gw + 1)) / nwarp;
    if (t >= t1) return;
    auto row_start = [&](long long A_) { return A_ * n - A_ * (A_ - 1) / 2; };
    int A = (int)(((double)(2 * n + 1) - sqrt((double)(2 * n + 1) * (double)(2 * n + 1) - 8.0 * (double)t)) * 0.5);
    if (A < 0) A = 0;
    if (A > nchunk - 1) A = nchunk - 1;
    while (A > 0 && row_start(A) > t) --A;
    while (A < nchunk - 1 && row_start(A + 1) <= t) ++A;
    int B = A + (int)(t - row_start(A));

    auto load_B = [&](int cB, int buf) {                          // whole warp: chunk cB -> buffer buf (asynchronous)
        const char* src = F32 ? reinterpret_cast<const char*>(w.pk32 + (size_t)cB * CHUNK)
                              : reinterpret_cast<const char*>(w.pk64 + (size_t)cB * CHUNK);
#pragma unroll
        for (int k = 0; k < CHUNK * Sm::POS_BYTES / 512; ++k) {
            const int piece = k * 32 + lane;                          // 16-byte pieces of the chunk, in memory order
            // FP64: body b = 2u + h is the pieces 2b (x, y) and 2b + 1 (z, G m); they go to plane 2h + (0 | 1), entry u,
            // so that lanes reading consecutive pairs u hit consecutive 16-byte words (no bank conflicts in the ring)
            const int dst = F32 ? piece : (piece & 3) * (CHUNK / 2) + (piece >> 2);
            cp_async16(&sm.pos[buf][dst * 16], src + (size_t)piece * 16);
        }
        if (lane < 3) cp_async16(reinterpret_cast<char*>(&sm.bcB[buf]) + 16 * lane, reinterpret_cast<const char*>(w.bc + cB) + 16 * lane);
        cp_async_commit();
    };
    auto flush_row = [&](int cA) {                                // stationary sums of chunk cA -> aslot[]
        double* g = w.aslot + (size_t)cA * CHUNK;
#pragma unroll
        for (int k = 0; k < CHUNK / 64; ++k) {
            const int u = lane + 32 * k;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (cA * CHUNK + 2 * u + h < N) {
                    atomicAdd(g + h * (CHUNK / 2) + u, sm.accS[0][2 * u + h]);
                    atomicAdd(g + NP + h * (CHUNK / 2) + u, sm.accS[1][2 * u + h]);
                    atomicAdd(g + 2 * NP + h * (CHUNK / 2) + u, sm.accS[2][2 * u + h]);
                }
            }
        }
    };

    int buf = 0;
    load_B(B, buf);
    int rowA = -1;
    double xi[P], yi[P], zi[P], gi64[P];                              // FP64 kernel: stationary bodies in registers
    float gi32[P];                                                    // FP32 kernel: their G m (positions: sm.xiS)
    while (t < t1) {
        if (A != rowA) {                                              // a new row: this warp's stationary chunk
            if (rowA >= 0) flush_row(rowA);
            rowA = A;
#pragma unroll
            for (int p = 0; p < P; ++p) {
                const int bi = 2 * (lane + 32 * (p >> 1)) + (p & 1);
                const double4 q = w.pk64[(size_t)A * CHUNK + bi];
                if constexpr (F32) {
                    sm.xiS[0][bi] = q.x; sm.xiS[1][bi] = q.y; sm.xiS[2][bi] = q.z;
                    gi32[p] = (float)q.w;
                } else {
                    xi[p] = q.x; yi[p] = q.y; zi[p] = q.z; gi64[p] = q.w;
                }
                sm.accS[0][bi] = 0.0; sm.accS[1][bi] = 0.0; sm.accS[2][bi] = 0.0;
            }
            if (lane == 0) sm.bcA = w.bc[A];
            __syncwarp();
        }
        // the tile after this one (same row, or the diagonal tile of the next row): start its copy now
        int A2 = A, B2 = B + 1;
        if (B2 >= nchunk) { A2 = A + 1; B2 = A2; }
        const bool more = t + 1 < t1;
        if (more) { load_B(B2, buf ^ 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        __syncwarp();

        const ChunkP& Ac = sm.bcA;
        const ChunkP& Bc = sm.bcB[buf];
        const int mode = (A == B) ? 2 : (tile_is_far(Ac, Bc) ? 0 : 1);
        const bool uni = Ac.uni != 0.f && Bc.uni != 0.f;              // both chunks uniform in mass: G m factored out of the pair loop
        double* aS = &sm.accS[0][0];
        double* gT = w.aslot + (size_t)B * CHUNK;
        if constexpr (F32) {
            const float4* pB = reinterpret_cast<const float4*>(&sm.pos[buf][0]);
            const double* xS = &sm.xiS[0][0];
            if (mode == 0 && uni) tile32<CHUNK, 0, true>(lane, pB, Ac, Bc, xS, gi32, aS, gT, NP, A, B, N, w, cand_cap);
            else if (mode == 0) tile32<CHUNK, 0>(lane, pB, Ac, Bc, xS, gi32, aS, gT, NP, A, B, N, w, cand_cap);
            else if (mode == 1) tile32<CHUNK, 1>(lane, pB, Ac, Bc, xS, gi32, aS, gT, NP, A, B, N, w, cand_cap);
            else                tile32<CHUNK, 2>(lane, pB, Ac, Bc, xS, gi32, aS, gT, NP, A, B, N, w, cand_cap);
        } else {
            const double2* pB = reinterpret_cast<const double2*>(&sm.pos[buf][0]);
            if (mode == 0 && uni) tile64<CHUNK, 0, true>(lane, pB, Ac, Bc, xi, yi, zi, gi64, aS, gT, NP, A, B, N, w, cand_cap);
            else if (mode == 0) tile64<CHUNK, 0>(lane, pB, Ac, Bc, xi, yi, zi, gi64, aS, gT, NP, A, B, N, w, cand_cap);
            else if (mode == 1) tile64<CHUNK, 1>(lane, pB, Ac, Bc, xi, yi, zi, gi64, aS, gT, NP, A, B, N, w, cand_cap);
            else                tile64<CHUNK, 2>(lane, pB, Ac, Bc, xi, yi, zi, gi64, aS, gT, NP, A, B, N, w, cand_cap);
        }
        __syncwarp();                                                 // buffer buf may be overwritten two tiles on
        ++t; A = A2; B = B2; buf ^= 1;
    }
    flush_row(rowA);
}

}  // namespace ksym
}  // namespace genga
