// Register-only arithmetic chains that measure this device's FP64 DFMA, FP64 tensor (mma.sync m8n8k4 f64 -> DMMA)
// and FP32 FFMA peaks: the roofline denominators bench.py reports K2, K3 and K5 against (SURVEY.md 8(d) "the builder
// must also measure a register-only DFMA/FFMA chain").  Eight independent dependent chains per thread, 8 warps per
// scheduler: enough to cover the pipe latency; no memory traffic inside the timed loop.
#include "se_common.cuh"

namespace {

constexpr int PEAK_ITERS = 4096;
constexpr int PEAK_CHAINS = 8;

template <typename T>
__global__ void __launch_bounds__(1024) k_peak_fma(T *out, T a, T b)
{
    T v[PEAK_CHAINS];
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) v[c] = (T)(threadIdx.x + c) * (T)1e-3;
#pragma unroll 16                                                 // 128 FMAs per loop-counter update and branch
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
        for (int c = 0; c < PEAK_CHAINS; ++c) v[c] = fma(v[c], a, b);
    }
    T s = 0;
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) s += v[c];
    if (s == (T)123456789) out[0] = s;                           // keeps the chains alive, never taken
}

__global__ void __launch_bounds__(1024) k_peak_dmma(double *out, double a, double b)
{
    double c[PEAK_CHAINS][2];
#pragma unroll
    for (int k = 0; k < PEAK_CHAINS; ++k) c[k][0] = c[k][1] = (double)(threadIdx.x + k) * 1e-3;
#pragma unroll 8
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
        for (int k = 0; k < PEAK_CHAINS; ++k)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[k][0]), "+d"(c[k][1])
                         : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int k = 0; k < PEAK_CHAINS; ++k) s += c[k][0] + c[k][1];
    if (s == 123456789.0) out[0] = s;
}

// read + write stream, 16 bytes per access, grid-stride
__global__ void __launch_bounds__(256) k_peak_stream(const float4 *in, float4 *out, size_t n)
{
    // four independent 16-byte loads in flight per thread and trip
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < n; i += 4 * stride) {
        float4 v0 = in[i], v1 = in[i + stride], v2 = in[i + 2 * stride], v3 = in[i + 3 * stride];
        v0.x += 1.0f; v1.x += 1.0f; v2.x += 1.0f; v3.x += 1.0f;
        out[i] = v0; out[i + stride] = v1; out[i + 2 * stride] = v2; out[i + 3 * stride] = v3;
    }
    for (; i < n; i += stride) {
        float4 v = in[i];
        v.x += 1.0f;
        out[i] = v;
    }
}

se_status measure_stream(int reps, int nsm, double *tbs)
{
    // in place, like K4 (every 16 bytes read once and written once to the same address)
    const size_t bytes = (size_t)1 << 31, n = bytes / sizeof(float4);
    float4 *a = nullptr;
    if (cudaMalloc(&a, bytes) != cudaSuccess) { cudaGetLastError(); return SE_ENOMEM; }
    float4 *b = a;
    cudaMemset(a, 0, bytes);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int r = 0; r < reps + 1; ++r) {
        cudaEventRecord(e0);
        k_peak_stream<<<nsm * 8, 256>>>(a, b, n);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(a);
    if (cudaGetLastError() != cudaSuccess || best > 1e29f) return SE_ECUDA;
    *tbs = 2.0 * (double)bytes / (best * 1e-3) / 1e12;
    return SE_OK;
}

}  // namespace

extern "C" se_status se_measure_peak(int which, int reps, double *tflops)
{
    if (!tflops || which < 0 || which > 3 || reps < 1) return SE_EINVAL;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return SE_ECUDA;
    }
    if (which == 3) return measure_stream(reps, nsm, tflops);
    double *out = nullptr;
    if (cudaMalloc(&out, 64) != cudaSuccess) { cudaGetLastError(); return SE_ENOMEM; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int threads = 1024, blocks = 2 * nsm;                  // 64 warps per SM
    // FMAs per thread: chains x iterations (DMMA: 256 FMA per warp instruction = 8 per thread)
    const double fma_per_thread = (double)PEAK_CHAINS * PEAK_ITERS * (which == 1 ? 8.0 : 1.0);
    float best = 1e30f;
    for (int r = 0; r < reps + 1; ++r) {
        cudaEventRecord(e0);
        if (which == 0) k_peak_fma<double><<<blocks, threads>>>(out, 0.999, 1e-3);
        else if (which == 1) k_peak_dmma<<<blocks, threads>>>(out, 0.5, 1e-3);
        else k_peak_fma<float><<<blocks, threads>>>((float *)out, 0.999f, 1e-3f);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms;                       // first launch is the warm-up
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    if (cudaGetLastError() != cudaSuccess || best > 1e29f) return SE_ECUDA;
    *tflops = 2.0 * fma_per_thread * threads * blocks / (best * 1e-3) / 1e12;
    return SE_OK;
}
