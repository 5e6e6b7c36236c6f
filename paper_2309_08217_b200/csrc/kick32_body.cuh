// kick32_body.cuh -- the all-pairs long-range kick in FP32 force precision (PAPER.md:19, 43, 223:
// "Do Kick in single precision = 1").
//
// a_i = sum_{j != i} G m_j (x_j - x_i) / r_ij^3 over FAR pairs, mixed-precision policy P32
// (DESIGN.md section 3): positions relative to the origin of each 128-body j-chunk (FP64
// subtraction, one rounding to FP32), packed FP32 arithmetic (FFMA2/FADD2/FMUL2: two j-bodies per
// instruction), MUFU.RSQ, FP32 partial sums over one chunk, chunk partials accumulated in FP64.
// A (body, chunk) whose smallest r^2 (own slot left out) is not above the conservative bound
// (lambda * r_crit upper bound, frame guard) is NOT added: it is pushed to the candidate list and
// re-evaluated pair by pair in FP64 with the changeover function by the near-field kernel
// (encounter forces always in FP64).  Chunks whose bounding sphere is out of reach of
// every body of the warp run a copy of the loop without the smallest-r^2 tracking.
//
// Layout: I i-bodies per thread (FP64 positions and bound parameters in shared memory); j-bodies
// streamed through shared memory in 1024-body stages by bulk asynchronous copies (cp.async.bulk ->
// UBLKCP, mbarrier completion, double buffered); one CTA owns a contiguous run of (i-block, chunk)
// units so that 148 x occupancy CTAs carry equal work.  Variants (genga_set_tuning / genga_autotune)
// differ in I, threads, registers, unroll, and plain vs mass-scaled j-records.
#pragma once

#include "tile_pipeline.cuh"

namespace genga {
namespace k32 {


typedef unsigned long long f2;   // two packed floats (lo = even j, hi = odd j)

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
__device__ __forceinline__ float min3(float a, float b, float c)
{
    float r; asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r;
}


// One j-chunk against the I i-bodies of this thread.  SELF: the chunk holds this warp's own
// slots; the self pair is then left out of the smallest-r^2 tracking (slot index compare), so a
// body's own chunk is flagged only if a DIFFERENT body is near.
template <int I, int UNR, bool SELF, bool SC, bool FAR, int CHUNK>
__device__ __forceinline__ void pair_loop(const float4* __restrict__ jp, const float (&nx)[I], const float (&ny)[I],
                                          const float (&nz)[I], f2 (&ax)[I], f2 (&ay)[I], f2 (&az)[I],
                                          float (&mn)[I], const int (&self_off)[I])
{
#pragma unroll UNR
    for (int jj = 0; jj < CHUNK / 2; ++jj) {
        const float4 A = jp[jj], B = jp[CHUNK / 2 + jj];     // planes (x0,x1,y0,y1) | (z0,z1,g0,g1)
        const f2 xj = pk(A.x, A.y), yj = pk(A.z, A.w), zj = pk(B.x, B.y), gj = pk(B.z, B.w);
#pragma unroll
        for (int k = 0; k < I; ++k) {
            // plain: d = x_j - x_i.  mass-scaled (SC): D = q_j x_j - q_j x_i with q = (G m)^(-1/2)
            const f2 dx = SC ? fma2(gj, pk(nx[k], nx[k]), xj) : add2(xj, pk(nx[k], nx[k]));
            const f2 dy = SC ? fma2(gj, pk(ny[k], ny[k]), yj) : add2(yj, pk(ny[k], ny[k]));
            const f2 dz = SC ? fma2(gj, pk(nz[k], nz[k]), zj) : add2(zj, pk(nz[k], nz[k]));
            f2 r2 = mul2(dx, dx);
            r2 = fma2(dy, dy, r2);
            r2 = fma2(dz, dz, r2);
            float r2a, r2b; upk(r2, r2a, r2b);
            float ya, yb;
            if (SELF) {
                const bool sa = (2 * jj == self_off[k]), sb = (2 * jj + 1 == self_off[k]);
                mn[k] = min3(mn[k], sa ? 3.0e38f : r2a, sb ? 3.0e38f : r2b);
                ya = rsq(r2a); yb = rsq(r2b);
                // the self term is 0 by selection, for any mass: d_self = 0 gives y = inf (plain records), and
                // D_self is rounding residue (mass-scaled records); a product with y would be NaN or garbage
                ya = sa ? 0.f : ya; yb = sb ? 0.f : yb;
            } else {
                if (!FAR) mn[k] = min3(mn[k], r2a, r2b);      // FAR: the chunk's bounding sphere is out of reach
                ya = rsq(r2a); yb = rsq(r2b);
            }
            const f2 y = pk(ya, yb);
            const f2 t = mul2(y, y);
            f2 s = SC ? mul2(t, y) : mul2(mul2(y, gj), t);       // SC: |D|^-3 = G m / r^3 / q
            ax[k] = fma2(s, dx, ax[k]);
            ay[k] = fma2(s, dy, ay[k]);
            az[k] = fma2(s, dz, az[k]);
        }
    }
}

// Kernel configuration: I i-bodies per thread, NT threads per CTA (I * NT = 512 = one i-block),
// MINB CTAs per SM asked of ptxas (caps the registers), ACCS: FP64 accumulators in shared memory
// instead of registers, UNR: unroll factor of the j-pair loop.
template <int I, int NT, bool ACCS, int CHUNK>
struct __align__(16) Smem32 {
    float4   j[NSTAGE][STAGE_J];                 // pair-interleaved j data (chunk-relative), 16 B per body
    ChunkP   bc[NSTAGE][STAGE_J / CHUNK];
    double   xi[3][I][NT];                       // FP64 positions of this CTA's i-bodies
    double   acc[ACCS ? 3 : 1][ACCS ? I : 1][ACCS ? NT : 1];   // FP64 accumulators (ACCS)
    float    bp[3][I][NT];                       // bound parameters (hq, aq, rf) of the i-bodies
    uint64_t full[NSTAGE];
};

// The whole kernel as a device function (smraw: sizeof(Smem32<...>) bytes of 16-byte aligned shared memory),
// so that the fused small-N step kernel (mega_step.cu) can run it as one of its phases.
template <int I, int NT, bool ACCS, int UNR, bool SC, int CHUNK>
__device__ __forceinline__ void kick32_body(int N, int nchunk, int nib, Workspace& w, unsigned int cand_cap,
                                            unsigned char* smraw)
{
    constexpr int BI = I * NT;
    static_assert(PAD_BODIES % BI == 0, "i-blocks tile the padding unit");
    constexpr int STAGE_CH = STAGE_J / CHUNK;      // chunks per shared-memory stage
    Smem32<I, NT, ACCS, CHUNK>& sm = *reinterpret_cast<Smem32<I, NT, ACCS, CHUNK>*>(smraw);
    const int tid = threadIdx.x;

    if (tid == 0) {
        for (int s = 0; s < NSTAGE; ++s) mbar_init(&sm.full[s], 1);
        fence_barrier_init();
    }
    __syncthreads();
    uint32_t phase = 0u;                           // bit b = parity of stage buffer b

    const long long U = (long long)nib * nchunk;
    long long u0 = (U * (long long)blockIdx.x) / (long long)gridDim.x;
    const long long u1 = (U * (long long)(blockIdx.x + 1)) / (long long)gridDim.x;

    while (u0 < u1) {
        const int ib = (int)(u0 / nchunk);
        const int c0 = (int)(u0 - (long long)ib * nchunk);
        const int c1 = (int)min((long long)nchunk, (long long)c0 + (u1 - u0));
        u0 += (c1 - c0);

        // ---- i-side: FP64 positions and bound parameters to shared memory (own column only)
        double Ax[ACCS ? 1 : I], Ay[ACCS ? 1 : I], Az[ACCS ? 1 : I];
#pragma unroll
        for (int k = 0; k < I; ++k) {
            const int i = ib * BI + k * NT + tid;
            const double4 q = w.pk64[i];
            sm.xi[0][k][tid] = q.x; sm.xi[1][k][tid] = q.y; sm.xi[2][k][tid] = q.z;
            const BoundP b = w.bi[i];
            sm.bp[0][k][tid] = b.hq; sm.bp[1][k][tid] = b.aq; sm.bp[2][k][tid] = b.rf;
            if (ACCS) { sm.acc[0][k][tid] = 0.0; sm.acc[1][k][tid] = 0.0; sm.acc[2][k][tid] = 0.0; }
            else      { Ax[k] = 0.0; Ay[k] = 0.0; Az[k] = 0.0; }
        }

        const int nst = (c1 - c0 + STAGE_CH - 1) / STAGE_CH;
        auto issue = [&](int st) {
            const int cs  = c0 + st * STAGE_CH;
            const int nch = min(STAGE_CH, c1 - cs);
            const int b   = st & 1;
            const uint32_t bytes_j = (uint32_t)nch * CHUNK * 16u;
            const uint32_t bytes_b = (uint32_t)nch * (uint32_t)sizeof(ChunkP);
            fence_proxy_async();
            mbar_expect_tx(&sm.full[b], bytes_j + bytes_b);
            bulk_g2s(&sm.j[b][0], w.pk32 + (size_t)cs * CHUNK, bytes_j, &sm.full[b]);
            bulk_g2s(&sm.bc[b][0], w.bc + cs, bytes_b, &sm.full[b]);
        };
        if (tid == 0) { issue(0); if (nst > 1) issue(1); }

        for (int st = 0; st < nst; ++st) {
            const int b   = st & 1;
            const int cs  = c0 + st * STAGE_CH;
            const int nch = min(STAGE_CH, c1 - cs);
            mbar_wait(&sm.full[b], (phase >> b) & 1u);
            phase ^= 1u << b;

            for (int ch = 0; ch < nch; ++ch) {
                const ChunkP& Bc = sm.bc[b][ch];
                // i-positions in the chunk's frame: FP64 subtraction, then one rounding to FP32
                float nx[I], ny[I], nz[I];
                f2 ax[I], ay[I], az[I];
                float mn[I];
                {
                    const double ox = Bc.ox, oy = Bc.oy, oz = Bc.oz;
#pragma unroll
                    for (int k = 0; k < I; ++k) {
                        nx[k] = (float)(ox - sm.xi[0][k][tid]);
                        ny[k] = (float)(oy - sm.xi[1][k][tid]);
                        nz[k] = (float)(oz - sm.xi[2][k][tid]);
                        ax[k] = 0ull; ay[k] = 0ull; az[k] = 0ull; mn[k] = 3.0e38f;
                    }
                }

                const float4* jp = &sm.j[b][ch * CHUNK];
                // offset of each own slot inside this chunk (outside [0, CHUNK) unless it is the own chunk);
                // warp-uniform decision: a warp's 32 slots of one k lie in one chunk
                int self_off[I];
                bool self = false;
#pragma unroll
                for (int k = 0; k < I; ++k) {
                    self_off[k] = ib * BI + k * NT + tid - (cs + ch) * CHUNK;
                    self = self || (self_off[k] >= 0 && self_off[k] < CHUNK);
                }
                // bound of this (body, chunk) and the sphere test: if every body of the warp is farther from the
                // chunk's frame origin than bound + chunk radius, no pair of the chunk can be near (triangle
                // inequality), and the loop without the smallest-r^2 tracking runs (one instruction less per two pairs)
                const float Hc = Bc.hq, Ac = Bc.aq, Rc = Bc.rf, Q2 = Bc.q2max, Rad = Bc.rad;
                float Bq[I];
                bool far = true;
#pragma unroll
                for (int k = 0; k < I; ++k) {
                    Bq[k] = fmaxf(fmaxf(sm.bp[0][k][tid], Hc) * fmaxf(sm.bp[1][k][tid], Ac), fmaxf(sm.bp[2][k][tid], Rc));
                    const float reach = (Bq[k] + Rad) * 1.000004f;
                    const float d2 = fmaf(nz[k], nz[k], fmaf(ny[k], ny[k], nx[k] * nx[k]));
                    far = far && ((d2 > reach * reach) || (ib * BI + k * NT + tid >= N));
                }
                far = __all_sync(0xffffffffu, far);
                if (self)     pair_loop<I, UNR, true, SC, false, CHUNK>(jp, nx, ny, nz, ax, ay, az, mn, self_off);
                else if (far) pair_loop<I, UNR, false, SC, true, CHUNK>(jp, nx, ny, nz, ax, ay, az, mn, self_off);
                else          pair_loop<I, UNR, false, SC, false, CHUNK>(jp, nx, ny, nz, ax, ay, az, mn, self_off);

                // ---- chunk end: keep the FP32 partial or hand the chunk to the near field ----
#pragma unroll
                for (int k = 0; k < I; ++k) {
                    const float bound = (ib * BI + k * NT + tid < N) ? (SC ? Bq[k] * Bq[k] * Q2 : Bq[k] * Bq[k]) : -1.0f;
                    const bool keep = mn[k] > bound;
                    float lo, hi;
                    upk(ax[k], lo, hi); const float px = lo + hi;
                    upk(ay[k], lo, hi); const float py = lo + hi;
                    upk(az[k], lo, hi); const float pz = lo + hi;
                    if (ACCS) {
                        if (keep) {
                            sm.acc[0][k][tid] += (double)px;
                            sm.acc[1][k][tid] += (double)py;
                            sm.acc[2][k][tid] += (double)pz;
                        }
                    } else {
                        Ax[k] += keep ? (double)px : 0.0;
                        Ay[k] += keep ? (double)py : 0.0;
                        Az[k] += keep ? (double)pz : 0.0;
                    }
                    const unsigned int bal = __ballot_sync(0xffffffffu, !keep);
                    if (bal)
                        push_candidates(bal, !keep, ib * BI + k * NT + tid, cs + ch,
                                        &w.ctr->cand_count, w.cand, cand_cap);
                }
            }
            __syncthreads();                       // every thread is done reading buffer b
            if (tid == 0 && st + 2 < nst) issue(st + 2);
        }

#pragma unroll
        for (int k = 0; k < I; ++k) {
            if (ib * BI + k * NT + tid < N) {
                const int i = w.order[ib * BI + k * NT + tid];     // slot -> body (API order)
                atomicAdd(&w.a[3 * i + 0], ACCS ? sm.acc[0][k][tid] : Ax[ACCS ? 0 : k]);
                atomicAdd(&w.a[3 * i + 1], ACCS ? sm.acc[1][k][tid] : Ay[ACCS ? 0 : k]);
                atomicAdd(&w.a[3 * i + 2], ACCS ? sm.acc[2][k][tid] : Az[ACCS ? 0 : k]);
            }
        }
    }
}

}  // namespace k32
}  // namespace genga
