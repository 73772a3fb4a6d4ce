// peak.cu -- FP64 roofline denominator: an all-SM kernel of independent DFMA chains.
// MEASURED_PEAKS.json has no fp64 entry, so bench.py measures the sustained DFMA rate of the same GPU in the
// same run and reports the render kernel against it.
#include "common.cuh"
#include <algorithm>

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

// the same FP64 pipe driven by mma.sync.m8n8k4.f64 (DMMA, 256 FMAs per warp instruction): 8 independent accumulator tiles
__global__ void __launch_bounds__(256) dmma_chain_kernel(double* out, int iters, double a, double b)
{
    double c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = threadIdx.x * 1e-3 + i;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[2 * u]), "+d"(c[2 * u + 1])
                         : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i];
    if (s == 123456.789) out[0] = s;
}

static int measure_one(bool dmma, int repeats, double* burst, double* sustained);

// FP64-pipe peak in FMA/s: the larger of the DFMA-chain and the DMMA-chain rates (both feed the same pipe)
int measure_fp64_peak(int repeats, double* burst, double* sustained)
{
    double b0 = 0, s0 = 0, b1 = 0, s1 = 0;
    int rc = measure_one(false, repeats, &b0, &s0);
    if (rc) return rc;
    rc = measure_one(true, repeats, &b1, &s1);
    if (rc) return rc;
    if (burst) *burst = std::max(b0, b1);
    if (sustained) *sustained = std::max(s0, s1);
    return E2E_OK;
}

static int measure_one(bool dmma, int repeats, double* burst, double* sustained)
{
    int dev = 0, sms = 0;
    E2E_CUDA(cudaGetDevice(&dev));
    E2E_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (repeats < 2) repeats = 2;
    if (repeats > 4096) repeats = 4096;
    double* d_out = nullptr;
    E2E_CUDA(cudaMalloc(&d_out, 8));
    std::vector<cudaEvent_t> ev(repeats + 1, nullptr);
    for (auto& e : ev) cudaEventCreate(&e);
    const int iters = 8192, threads = 256, blocks = sms * 8;
    // FMAs per launch: 64 DFMAs per thread and iteration, or 8 DMMAs (256 FMAs each) per warp and iteration
    const double work = (double)blocks * threads * (double)iters * 64.0;
    auto launch = [&] {
        if (dmma) dmma_chain_kernel<<<blocks, threads>>>(d_out, iters, 0.999999, 1e-7);
        else dfma_chain_kernel<<<blocks, threads>>>(d_out, iters, 0.999999, 1e-7);
        count_launch();
    };
    launch();                                                                   // warm-up
    cudaEventRecord(ev[0]);
    for (int r = 0; r < repeats; ++r) {
        launch();
        cudaEventRecord(ev[r + 1]);
    }
    cudaError_t e = cudaEventSynchronize(ev[repeats]);
    double best = 0.0, sus = 0.0;
    if (e == cudaSuccess) {
        for (int r = 0; r < repeats; ++r) {
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ev[r], ev[r + 1]);
            if (ms > 0.f) best = std::max(best, work / (ms * 1e-3));
        }
        float ms = 0.f;
        const int h = repeats / 2;
        cudaEventElapsedTime(&ms, ev[h], ev[repeats]);
        if (ms > 0.f) sus = work * (repeats - h) / (ms * 1e-3);
    }
    for (auto& x : ev) cudaEventDestroy(x);
    cudaFree(d_out);
    if (e != cudaSuccess) return fail_cuda(e, "dfma_chain_kernel");
    if (burst) *burst = best;
    if (sustained) *sustained = sus;
    return E2E_OK;
}

}  // namespace e2e
