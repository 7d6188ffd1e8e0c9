// peak_kernels.cu -- measured FP32 FMA peak of the device (the "alu" roofline of the fp32 pair kernel
// is the MEASURED rate of a chain of independent fused multiply-adds, not the nominal lanes x clock figure).
#include "common.cuh"

namespace {

// every thread runs 16 independent FMA chains (enough to cover the 4-cycle latency with 8+ warps per scheduler)
__global__ void __launch_bounds__(512) fma_chain_kernel(float *out, int iters, float a, float b)
{
    float x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = (float)(threadIdx.x + i) * 1e-3f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == 123.456f) out[0] = s;   // keeps the chains alive
}

}  // namespace

extern "C" int pimd_measure_fp32_fma_tflops(void *cuda_stream, double *h_tflops)
{
    if (!h_tflops) { pimd_set_error("null argument"); return PIMD_ERR_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    PIMD_CUDA_CHECK(cudaGetDevice(&dev));
    PIMD_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float *d = nullptr;
    PIMD_CUDA_CHECK(cudaMalloc(&d, 64));   // (measurement helper outside any context: the only allocation the library ever makes)
    cudaEvent_t e0, e1;
    PIMD_CUDA_CHECK(cudaEventCreate(&e0));
    PIMD_CUDA_CHECK(cudaEventCreate(&e1));
    const int iters = 4096, blocks = sms * 4, threads = 512;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {       // first repetitions warm the clocks up
        cudaEventRecord(e0, st);
        fma_chain_kernel<<<blocks, threads, 0, st>>>(d, iters, 0.999f, 1e-3f);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 16.0 * (double)iters * (double)blocks * (double)threads;
        if (ms > 0.f) best = fmax(best, flops / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    PIMD_CUDA_CHECK(cudaGetLastError());
    *h_tflops = best;
    return 0;
}
