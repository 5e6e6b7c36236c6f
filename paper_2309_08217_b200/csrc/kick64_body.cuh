// kick64_body.cuh -- the all-pairs long-range kick in FP64 (GENGA's default).
//
// a_i = sum_{j != i} G m_j (x_j - x_i) / r_ij^3 over pairs OUTSIDE the changeover zone, every
// operation in FP64.  1/r^3 comes from the 20-bit MUFU.RSQ64H seed y0 and one cubic correction:
//   t = y0^2, e = 1 - r^2 t, 1/r^3 = y0^3 (1 - e)^(-3/2) = y0^3 (1 + 3/2 e + 15/8 e^2) + O(e^3),
// |e| <~ 2^-19 so the truncation is < 1e-17 relative.  16 FP64-pipe
// instructions per pair.  A (body, 128-j chunk) whose smallest r^2 (own slot left out) is not above the conservative
// r_crit bound is not added but handed to the near-field kernel, which applies K pair by pair.
#pragma once

#include "tile_pipeline.cuh"

namespace genga {
namespace k64 {


__device__ __forceinline__ double rsq64h(double a)
{
    double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r;
}

constexpr double EPS2 = 1.0e-60;   // added to r^2 so that the self pair (d = 0 exactly) contributes 0, not NaN;
                                   // changes no pair with r > 1e-22 au by even one ulp

// One j-chunk against the I i-bodies of this thread.  SELF: the chunk holds this warp's own slots;
// the self pair is left out of the smallest-r^2 tracking, so a body's own chunk is flagged only if
// a DIFFERENT body is near.  mn tracks the high word of r^2 (orders like r^2 >= 0).
template <int I, int UNR, bool SELF, bool FAR, int CHUNK>
__device__ __forceinline__ void pair_loop(const double4* __restrict__ jp, const double (&xi)[I], const double (&yi)[I],
                                          const double (&zi)[I], double (&ax)[I], double (&ay)[I], double (&az)[I],
                                          int (&mn)[I], const int (&self_off)[I])
{
#pragma unroll UNR
    for (int jj = 0; jj < CHUNK; ++jj) {
        const double4 J = jp[jj];
#pragma unroll
        for (int k = 0; k < I; ++k) {
            const double dx = J.x - xi[k];
            const double dy = J.y - yi[k];
            const double dz = J.z - zi[k];
            double r2 = SELF ? fma(dx, dx, EPS2) : dx * dx;
            r2 = fma(dy, dy, r2);
            r2 = fma(dz, dz, r2);
            if (SELF) mn[k] = min(mn[k], (jj == self_off[k]) ? 0x7fffffff : __double2hiint(r2));
            else if (!FAR) mn[k] = min(mn[k], __double2hiint(r2));   // FAR: the chunk's bounding sphere is out of reach
            const double y0 = rsq64h(r2);
            const double t  = y0 * y0;
            const double e  = fma(-r2, t, 1.0);
            const double c  = fma(1.875, e, 1.5);
            const double q  = (J.w * y0) * t;
            const double qe = q * e;
            const double s  = fma(qe, c, q);
            ax[k] = fma(s, dx, ax[k]);
            ay[k] = fma(s, dy, ay[k]);
            az[k] = fma(s, dz, az[k]);
        }
    }
}

template <int I, int NT, int CHUNK>
struct __align__(16) Smem64 {
    double4  j[NSTAGE][STAGE_J];                 // (x, y, z, G m), 32 B per body
    ChunkP   bc[NSTAGE][STAGE_J / CHUNK];
    float    bp[3][I][NT];                       // bound parameters (hq, aq, rf) of this CTA's i-bodies
    uint64_t full[NSTAGE];
};

// The whole kernel as a device function (smraw: sizeof(Smem64<...>) bytes of 16-byte aligned shared memory).
template <int I, int NT, int UNR, int CHUNK>
__device__ __forceinline__ void kick64_body(int N, int nchunk, int nib, Workspace& w, unsigned int cand_cap,
                                            unsigned char* smraw)
{
    constexpr int BI = I * NT;
    static_assert(PAD_BODIES % BI == 0, "i-blocks tile the padding unit");
    constexpr int STAGE_CH = STAGE_J / CHUNK;      // chunks per shared-memory stage
    Smem64<I, NT, CHUNK>& sm = *reinterpret_cast<Smem64<I, NT, CHUNK>*>(smraw);
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

        double xi[I], yi[I], zi[I];
        double Ax[I], Ay[I], Az[I];
#pragma unroll
        for (int k = 0; k < I; ++k) {
            const int i = ib * BI + k * NT + tid;
            const double4 q = w.pk64[i];
            xi[k] = q.x; yi[k] = q.y; zi[k] = q.z;
            const BoundP b = w.bi[i];
            sm.bp[0][k][tid] = b.hq; sm.bp[1][k][tid] = b.aq; sm.bp[2][k][tid] = b.rf;
            Ax[k] = 0.0; Ay[k] = 0.0; Az[k] = 0.0;
        }

        const int nst = (c1 - c0 + STAGE_CH - 1) / STAGE_CH;
        auto issue = [&](int st) {
            const int cs  = c0 + st * STAGE_CH;
            const int nch = min(STAGE_CH, c1 - cs);
            const int b   = st & 1;
            const uint32_t bytes_j = (uint32_t)nch * CHUNK * 32u;
            const uint32_t bytes_b = (uint32_t)nch * (uint32_t)sizeof(ChunkP);
            fence_proxy_async();
            mbar_expect_tx(&sm.full[b], bytes_j + bytes_b);
            bulk_g2s(&sm.j[b][0], w.pk64 + (size_t)cs * CHUNK, bytes_j, &sm.full[b]);
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
                const ChunkP Bc = sm.bc[b][ch];
                double ax[I], ay[I], az[I];
                int mn[I];                        // high word of the smallest r^2 (orders like r^2 >= 0)
#pragma unroll
                for (int k = 0; k < I; ++k) { ax[k] = 0.0; ay[k] = 0.0; az[k] = 0.0; mn[k] = 0x7fffffff; }

                const double4* jp = &sm.j[b][ch * CHUNK];
                int self_off[I];                  // offset of each own slot inside this chunk (warp-uniform range test)
                bool self = false;
#pragma unroll
                for (int k = 0; k < I; ++k) {
                    self_off[k] = ib * BI + k * NT + tid - (cs + ch) * CHUNK;
                    self = self || (self_off[k] >= 0 && self_off[k] < CHUNK);
                }
                // sphere test (as in the FP32 kernel): every body of the warp farther from the chunk's frame origin
                // than bound + chunk radius => no near pair in this chunk, the loop without the min tracking runs
                float Bqk[I];
                bool far = true;
#pragma unroll
                for (int k = 0; k < I; ++k) {
                    Bqk[k] = fmaxf(fmaxf(sm.bp[0][k][tid], Bc.hq) * fmaxf(sm.bp[1][k][tid], Bc.aq),
                                   fmaxf(sm.bp[2][k][tid], Bc.rf));
                    const double reach = ((double)Bqk[k] + (double)Bc.rad) * 1.000001;
                    const double ex = xi[k] - Bc.ox, ey = yi[k] - Bc.oy, ez = zi[k] - Bc.oz;
                    const double d2 = fma(ez, ez, fma(ey, ey, ex * ex));
                    far = far && ((d2 > reach * reach) || (ib * BI + k * NT + tid >= N));
                }
                far = __all_sync(0xffffffffu, far);
                if (self)     pair_loop<I, UNR, true, false, CHUNK>(jp, xi, yi, zi, ax, ay, az, mn, self_off);
                else if (far) pair_loop<I, UNR, false, true, CHUNK>(jp, xi, yi, zi, ax, ay, az, mn, self_off);
                else          pair_loop<I, UNR, false, false, CHUNK>(jp, xi, yi, zi, ax, ay, az, mn, self_off);

#pragma unroll
                for (int k = 0; k < I; ++k) {
                    const float Bq = Bqk[k];
                    // bound in FP64, rounded up by one FP32 ulp-ish factor; compare high words only:
                    // equal high words count as "near" (conservative).
                    const double bd = (double)Bq * (double)Bq * 1.000001;
                    const int bh = (ib * BI + k * NT + tid < N) ? __double2hiint(bd) : -1;
                    const bool keep = mn[k] > bh;
                    Ax[k] += keep ? ax[k] : 0.0;
                    Ay[k] += keep ? ay[k] : 0.0;
                    Az[k] += keep ? az[k] : 0.0;
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
                atomicAdd(&w.a[3 * i + 0], Ax[k]);
                atomicAdd(&w.a[3 * i + 1], Ay[k]);
                atomicAdd(&w.a[3 * i + 2], Az[k]);
            }
        }
    }
}

}  // namespace k64
}  // namespace genga
