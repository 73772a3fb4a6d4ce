// peak.cu -- FP64 roofline denominator: an all-SM kernel of independent DFMA chains.
// MEASURED_PEAKS.json has no fp64 entry, so bench.py measures the sustained DFMA rate of the same GPU in the
// same run and reports the render kernel against it.
#include "common.cuh"

namespace e2e {

__global__ void __launch_bounds__(256) dfma_chain_kernel(double* out, int iters, double a, double b)
{
    double x0 = threadIdx.x * 1e-3, x1 = x0 + 0.1, x2 = x0 + 0.2, x3 = x0 + 0.3;
    double x4 = x0 + 0.4, x5 = x0 + 0.5, x6 = x0 + 0.6, x7 = x0 + 0.7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123456.789) out[0] = s;      // never true: keeps the chains alive
}

int measure_fp64_peak(int repeats, double* dfma_per_s, double* ms_out)
{
    int dev = 0, sms = 0;
    E2E_CUDA(cudaGetDevice(&dev));
    E2E_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* d_out = nullptr;
    E2E_CUDA(cudaMalloc(&d_out, 8));
    cudaEvent_t e0, e1;
    E2E_CUDA(cudaEventCreate(&e0));
    E2E_CUDA(cudaEventCreate(&e1));
    const int iters = 8192, threads = 256, blocks = sms * 8;
    double best = 0.0, best_ms = 0.0;
    for (int r = 0; r < (repeats < 1 ? 1 : repeats) + 1; ++r) {
        cudaEventRecord(e0);
        dfma_chain_kernel<<<blocks, threads>>>(d_out, iters, 0.999999, 1e-7);
        count_launch();
        cudaEventRecord(e1);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(d_out); return fail_cuda(e, "dfma_chain_kernel"); }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double rate = (double)blocks * threads * (double)iters * 64.0 / (ms * 1e-3);
        if (r > 0 && rate > best) { best = rate; best_ms = ms; }   // first run is warm-up
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    if (dfma_per_s) *dfma_per_s = best;
    if (ms_out) *ms_out = best_ms;
    return E2E_OK;
}

}  // namespace e2e
