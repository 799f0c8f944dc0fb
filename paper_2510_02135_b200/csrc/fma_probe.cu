// fma_probe.cu -- measurement helper for bench.py, built as its own library (liblm_probe.so): NOT part of liblm.so.
// Register-only FFMA2 / DFMA loops that measure the FMA-pipe peak of the current device in lane-operations per
// second (one lane-op = one fp32 / fp64 FMA on one lane): the roofline denominator bench.py reports next to the
// nominal one.
#include <cuda_runtime.h>

#include <algorithm>

namespace {

__global__ void probe_ffma2_kernel(float* out, float a, float b, int iters)
{
    float2 x[8];
    const float2 aa = make_float2(a, a), bb = make_float2(b, b);
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = make_float2(threadIdx.x * 1e-3f + i, (float)i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = __ffma2_rn(x[i], aa, bb);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i].x + x[i].y;
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void probe_dfma_kernel(double* out, double a, double b, int iters)
{
    double x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

// precision: 0 = fp32 (FFMA2), 1 = fp64 (DFMA).  Runs for about `seconds`; best launch wins.  Returns 0, or -1 on
// a bad argument / -5 on a CUDA error (the LM_E_* values of include/lm.h).
extern "C" int lm_probe_fma_peak(int precision, double seconds, double* lane_ops_per_s)
{
    if (!lane_ops_per_s) return -4;
    if (precision != 0 && precision != 1) return -1;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -5;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -5;
    const int threads = 256, grid = sms * 8, iters = 8192;
    void* buf = nullptr;
    if (cudaMalloc(&buf, (size_t)grid * threads * 8) != cudaSuccess) return -5;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    auto launch = [&]() {
        if (precision == 0) probe_ffma2_kernel<<<grid, threads>>>((float*)buf, 1.0001f, 0.5f, iters);
        else probe_dfma_kernel<<<grid, threads>>>((double*)buf, 1.0001, 0.5, iters);
    };
    const double ops_per_launch = (double)grid * threads * iters * (precision == 0 ? 16.0 : 8.0);
    launch();
    launch();
    cudaDeviceSynchronize();
    double best = 0.0, elapsed = 0.0;
    int reps = 0;
    while (elapsed < seconds * 1e3 || reps < 3) {
        cudaEventRecord(e0);
        launch();
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        elapsed += ms;
        best = std::max(best, ops_per_launch / (ms * 1e-3));
        if (++reps > 100000) break;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    if (cudaGetLastError() != cudaSuccess) return -5;
    *lane_ops_per_s = best;
    return 0;
}
