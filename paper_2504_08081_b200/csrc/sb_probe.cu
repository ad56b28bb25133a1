// sb_probe.cu -- measurement utility: FP32 FMA-chain microbenchmark (the roofline denominator
// of an ALU-bound path; MEASURED_PEAKS.json has no FP32 CUDA-core figure).  C ABI, no torch.
//   sbp_fma_peak: 8 independent FFMA chains per thread, full occupancy (2 x 1024 threads per SM),
//   timed with CUDA events on the given stream.  flops = threads * iters * 8 chains * 2.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {
__global__ void __launch_bounds__(1024, 2) fma_chain_kernel(float *out, int iters, float a, float b)
{
    float x0 = threadIdx.x * 1e-3f, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f;
    float x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    float s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == 12345.678f) out[blockIdx.x * blockDim.x + threadIdx.x] = s; // keep the chains alive
}
} // namespace

extern "C" {

// Returns 0 on success.  *out_tflops = best of `reps` timed launches; *out_ms = its duration.
int sbp_fma_peak(int iters, int reps, void *stream, double *out_tflops, double *out_ms)
{
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
    cudaStream_t st = (cudaStream_t)stream;
    const int blocks = n_sm * 2 * 4, threads = 1024;
    float *buf = nullptr;
    if (cudaMalloc(&buf, sizeof(float) * (size_t)blocks * threads) != cudaSuccess) return -2;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    fma_chain_kernel<<<blocks, threads, 0, st>>>(buf, iters, 0.999f, 1e-3f); // warm-up
    double best = 1e30;
    for (int r = 0; r < reps; ++r) {
        cudaEventRecord(e0, st);
        fma_chain_kernel<<<blocks, threads, 0, st>>>(buf, iters, 0.999f, 1e-3f);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(buf); return -3; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    const double flops = (double)blocks * threads * (double)iters * 16.0 * 8.0 * 2.0;
    if (out_ms) *out_ms = best;
    if (out_tflops) *out_tflops = flops / (best * 1e-3) * 1e-12;
    return 0;
}

} // extern "C"
