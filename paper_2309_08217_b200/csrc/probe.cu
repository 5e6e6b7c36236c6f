// probe.cu -- ALU peak probes: register-only instruction streams on every SM, used to put the
// measured FP32 / FP64 / MUFU issue rates of this B200 beside the nominal peaks that the roofline
// fractions are quoted against.  Not on the hot path.
#include "genga_internal.cuh"

namespace genga {

namespace {

typedef unsigned long long f2;
__device__ __forceinline__ f2 pk(float lo, float hi)
{
    f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r;
}
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c)
{
    f2 r; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r;
}

constexpr int CH = 8;        // independent chains per thread

__global__ void __launch_bounds__(256) probe_ffma(int iters, float* out)
{
    float a[CH];
    const float b = 1.0000001f, c = 1.0e-9f + threadIdx.x * 1e-12f;
#pragma unroll
    for (int k = 0; k < CH; ++k) a[k] = 1.0f + k + threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int k = 0; k < CH; ++k) a[k] = fmaf(a[k], b, c);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < CH; ++k) s += a[k];
    if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(256) probe_ffma2(int iters, float* out)
{
    f2 a[CH];
    const f2 b = pk(1.0000001f, 1.0000002f), c = pk(1.0e-9f + threadIdx.x * 1e-12f, 2.0e-9f);
#pragma unroll
    for (int k = 0; k < CH; ++k) a[k] = pk(1.0f + k + threadIdx.x, 2.0f + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int k = 0; k < CH; ++k) a[k] = fma2(a[k], b, c);
    }
    f2 s = 0ull;
#pragma unroll
    for (int k = 0; k < CH; ++k) s ^= a[k];
    if (s == 0x123456789abcdefull) out[0] = 1.f;
}

__global__ void __launch_bounds__(256) probe_dfma(int iters, double* out)
{
    double a[CH];
    const double b = 1.0000001, c = 1.0e-9 + threadIdx.x * 1e-12;
#pragma unroll
    for (int k = 0; k < CH; ++k) a[k] = 1.0 + k + threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int k = 0; k < CH; ++k) a[k] = fma(a[k], b, c);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < CH; ++k) s += a[k];
    if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(256) probe_rsq(int iters, float* out)
{
    float a[CH];
#pragma unroll
    for (int k = 0; k < CH; ++k) a[k] = 1.0f + k + threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int k = 0; k < CH; ++k) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < CH; ++k) s += a[k];
    if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(256) probe_rsq64h(int iters, double* out)
{
    double a[CH];
#pragma unroll
    for (int k = 0; k < CH; ++k) a[k] = 1.0 + k + threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int k = 0; k < CH; ++k) asm volatile("rsqrt.approx.ftz.f64 %0, %0;" : "+d"(a[k]));
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < CH; ++k) s += a[k];
    if (s == 123.456) out[0] = s;
}

// The FP32 pair loop of kick32_kernel on its own: j data read from shared memory (one 512-body
// stage, re-read), two i-bodies per thread, no staging, no per-chunk epilogue.  What the SM delivers
// for this instruction mix (12 packed-FP32 lane-ops + 1 MUFU + 1/2 FMNMX3 per pair) is the practical
// ceiling of the all-pairs kernel.  Counts pairs, reported through ops_per_s.
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f2 fma2n(f2 a, f2 b, f2 c) { f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ float rsqf(float a) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ float min3f(float a, float b, float c) { float r; asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r; }

template <bool WITH_MUFU, bool WITH_MIN, bool SC, int I, int UNR, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) probe_pairloop(int iters, float* out)
{
    __shared__ float4 sj[512];
    for (int q = threadIdx.x; q < 512; q += NT)
        sj[q] = make_float4(1.0f + q, 2.0f + 0.5f * q, 0.25f * q, 1.0e-3f);
    __syncthreads();
    float nx[I], ny[I], nz[I], mn[I];
    f2 ax[I], ay[I], az[I];
    for (int k = 0; k < I; ++k) {
        nx[k] = -0.37f * (threadIdx.x + 1 + k); ny[k] = 0.11f * threadIdx.x - k; nz[k] = 0.01f * k;
        ax[k] = 0ull; ay[k] = 0ull; az[k] = 0ull; mn[k] = 3.0e38f;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll UNR
        for (int jj = 0; jj < 256; ++jj) {
            const float4 A = sj[2 * jj], B = sj[2 * jj + 1];
            const f2 xj = pk(A.x, A.y), yj = pk(A.z, A.w), zj = pk(B.x, B.y), gj = pk(B.z, B.w);
#pragma unroll
            for (int k = 0; k < I; ++k) {
                const f2 dx = SC ? fma2n(gj, pk(nx[k], nx[k]), xj) : add2(xj, pk(nx[k], nx[k]));
                const f2 dy = SC ? fma2n(gj, pk(ny[k], ny[k]), yj) : add2(yj, pk(ny[k], ny[k]));
                const f2 dz = SC ? fma2n(gj, pk(nz[k], nz[k]), zj) : add2(zj, pk(nz[k], nz[k]));
                f2 r2 = mul2(dx, dx);
                r2 = fma2n(dy, dy, r2);
                r2 = fma2n(dz, dz, r2);
                float r2a, r2b;
                asm("mov.b64 {%0, %1}, %2;" : "=f"(r2a), "=f"(r2b) : "l"(r2));
                if (WITH_MIN) mn[k] = min3f(mn[k], r2a, r2b);
                const f2 y = WITH_MUFU ? pk(rsqf(r2a), rsqf(r2b)) : r2;
                const f2 t = mul2(y, y);
                const f2 s = SC ? mul2(t, y) : mul2(mul2(y, gj), t);
                ax[k] = fma2n(s, dx, ax[k]);
                ay[k] = fma2n(s, dy, ay[k]);
                az[k] = fma2n(s, dz, az[k]);
            }
        }
    }
    f2 sacc = 0ull; float sm = 0.f;
    for (int k = 0; k < I; ++k) { sacc ^= ax[k] ^ ay[k] ^ az[k]; sm += mn[k]; }
    if (sacc == 0x123456789abcdefull || sm == 123.456f) out[0] = 1.f;
}

}  // namespace

int run_peak_probe(int which, int iters, cudaStream_t s, double* ops_per_s, double* ms_out)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return GENGA_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return GENGA_ECUDA;
    if (iters < 1) iters = 1;
    const int blocks = sms * 8, threads = 256;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return GENGA_ECUDA;
    double best = 1e30;
    for (int rep = 0; rep < 4; ++rep) {            // first repetition is the warm-up
        cudaEventRecord(e0, s);
        switch (which) {
            case 0: probe_ffma<<<blocks, threads, 0, s>>>(iters, nullptr); break;
            case 1: probe_ffma2<<<blocks, threads, 0, s>>>(iters, nullptr); break;
            case 2: probe_dfma<<<blocks, threads, 0, s>>>(iters, nullptr); break;
            case 3: probe_rsq<<<blocks, threads, 0, s>>>(iters, nullptr); break;
            case 4: probe_rsq64h<<<blocks, threads, 0, s>>>(iters, nullptr); break;
            case 5: probe_pairloop<true, true, false, 2, 2, 256, 2><<<sms * 2, 256, 0, s>>>(iters, nullptr); break;
            case 6: probe_pairloop<false, true, false, 2, 2, 256, 2><<<sms * 2, 256, 0, s>>>(iters, nullptr); break;
            case 7: probe_pairloop<true, false, false, 2, 2, 256, 2><<<sms * 2, 256, 0, s>>>(iters, nullptr); break;
            case 8: probe_pairloop<true, true, true, 2, 2, 256, 2><<<sms * 2, 256, 0, s>>>(iters, nullptr); break;
            case 9: probe_pairloop<true, true, true, 2, 4, 256, 2><<<sms * 2, 256, 0, s>>>(iters, nullptr); break;
            case 10: probe_pairloop<true, false, true, 2, 4, 256, 2><<<sms * 2, 256, 0, s>>>(iters, nullptr); break;
            case 11: probe_pairloop<true, false, true, 4, 2, 128, 4><<<sms * 4, 128, 0, s>>>(iters, nullptr); break;
            case 12: probe_pairloop<true, false, true, 4, 2, 128, 3><<<sms * 3, 128, 0, s>>>(iters, nullptr); break;
            case 13: probe_pairloop<true, true, true, 4, 2, 128, 3><<<sms * 3, 128, 0, s>>>(iters, nullptr); break;
            case 14: probe_pairloop<false, false, true, 2, 4, 256, 2><<<sms * 2, 256, 0, s>>>(iters, nullptr); break;
            case 15: probe_pairloop<true, true, false, 2, 4, 256, 2><<<sms * 2, 256, 0, s>>>(iters, nullptr); break;
            case 16: probe_pairloop<true, true, true, 1, 8, 256, 4><<<sms * 4, 256, 0, s>>>(iters, nullptr); break;
            default: cudaEventDestroy(e0); cudaEventDestroy(e1); return GENGA_EINVAL;
        }
        cudaEventRecord(e1, s);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return GENGA_ECUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    double lane_ops = (double)blocks * threads * (double)iters * 8.0 * CH * ((which == 1) ? 2.0 : 1.0);
    if (which >= 5) {                                   // pairs = threads x i-bodies x 512 j x iters
        static const int thr_i[] = {512 * 2, 512 * 2, 512 * 2, 512 * 2, 512 * 2, 512 * 2, 512 * 4, 384 * 4, 384 * 4, 512 * 2, 512 * 2, 1024 * 1};
        lane_ops = (double)sms * thr_i[which - 5] * (double)iters * 512.0;
    }
    if (ops_per_s) *ops_per_s = lane_ops / (best * 1.0e-3);
    if (ms_out) *ms_out = best;
    return GENGA_OK;
}

}  // namespace genga
