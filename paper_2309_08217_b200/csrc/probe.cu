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
            default: cudaEventDestroy(e0); cudaEventDestroy(e1); return GENGA_EINVAL;
        }
        cudaEventRecord(e1, s);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return GENGA_ECUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    const double lane_ops = (double)blocks * threads * (double)iters * 8.0 * CH * ((which == 1) ? 2.0 : 1.0);
    if (ops_per_s) *ops_per_s = lane_ops / (best * 1.0e-3);
    if (ms_out) *ms_out = best;
    return GENGA_OK;
}

}  // namespace genga
