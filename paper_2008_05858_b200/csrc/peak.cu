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

// ------------------------------------------------------------------------------------------------
// e2e_probe_fp64_pipe: how the FP64 pipe of one SM behaves under the render kernel's instruction mix
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void probe_dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// one warp, NCH independent accumulator chains of DMMAs: cycles per round of NCH
template <int NCH>
__global__ void probe_chain_kernel(double* out, long long* cyc, int iters, double a, double b)
{
    double c[NCH][2];
#pragma unroll
    for (int i = 0; i < NCH; ++i) { c[i][0] = threadIdx.x + i; c[i][1] = 1.0; }
    const long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < NCH; ++u) probe_dmma(c[u][0], c[u][1], a, b);
    }
    const long long t1 = clock64();
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < NCH; ++i) s += c[i][0] + c[i][1];
    if (s == 1234.5) out[0] = s;
    if (threadIdx.x == 0) cyc[0] = t1 - t0;
}

// one CTA on one SM for a fixed number of cycles: warps [0, nd) issue DMMAs (4 chains each), warps [nd, nd + ns) issue
// independent scalar DFMAs (8 chains each); counts what each kind got done
__global__ void probe_mix_kernel(double* out, unsigned long long* cnt, int nd, int ns, long long cycles, double a, double b)
{
    const int w = threadIdx.x >> 5;
    const long long t0 = clock64();
    unsigned long long n = 0;
    if (w < nd) {
        double c[4][2] = {{1, 2}, {3, 4}, {5, 6}, {7, 8}};
        while (clock64() - t0 < cycles) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int u = 0; u < 4; ++u) probe_dmma(c[u][0], c[u][1], a, b);
            n += 32;
        }
        if (c[0][0] + c[1][0] + c[2][1] + c[3][1] == 1234.5) out[0] = 1.0;
        if ((threadIdx.x & 31) == 0) atomicAdd(&cnt[0], n);
    } else if (w < nd + ns) {
        double x[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = threadIdx.x + i;
        while (clock64() - t0 < cycles) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int u = 0; u < 8; ++u) x[u] = fma(x[u], a, b);
            n += 64;
        }
        double s = 0.0;
#pragma unroll
        for (int i = 0; i < 8; ++i) s += x[i];
        if (s == 1234.5) out[0] = s;
        if ((threadIdx.x & 31) == 0) atomicAdd(&cnt[1], n);
    }
}

int probe_fp64_pipe(double* r)
{
    double* d_out = nullptr;
    unsigned long long* d_cnt = nullptr;
    E2E_CUDA(cudaMalloc(&d_out, 8));
    cudaError_t e = cudaMalloc(&d_cnt, 16);
    if (e != cudaSuccess) { cudaFree(d_out); return fail_cuda(e, "probe_fp64_pipe: cudaMalloc"); }
    long long* d_cyc = reinterpret_cast<long long*>(d_cnt);
    const int iters = 4096;
    long long h = 0;
    probe_chain_kernel<1><<<1, 32>>>(d_out, d_cyc, iters, 0.999, 1e-7);
    probe_chain_kernel<1><<<1, 32>>>(d_out, d_cyc, iters, 0.999, 1e-7);
    cudaMemcpy(&h, d_cyc, 8, cudaMemcpyDeviceToHost);
    r[0] = (double)h / iters;                                   // cycles per DMMA, one dependent chain
    probe_chain_kernel<2><<<1, 32>>>(d_out, d_cyc, iters, 0.999, 1e-7);
    cudaMemcpy(&h, d_cyc, 8, cudaMemcpyDeviceToHost);
    r[1] = (double)h / iters / 2.0;                             // cycles per DMMA, two independent chains in one warp
    const long long cycles = 2000000;
    unsigned long long c[2];
    auto mix = [&](int nd, int ns, double& dm, double& sf) {
        cudaMemset(d_cnt, 0, 16);
        probe_mix_kernel<<<1, 32 * (nd + ns)>>>(d_out, d_cnt, nd, ns, cycles, 0.999, 1e-7);
        cudaMemcpy(c, d_cnt, 16, cudaMemcpyDeviceToHost);
        dm = (double)c[0] / (double)cycles; sf = (double)c[1] / (double)cycles;
    };
    double dm, sf;
    mix(16, 0, dm, sf); r[2] = dm;                              // DMMA per clock and SM, 16 DMMA warps alone (0.25 = the pipe's rate)
    mix(0, 4, dm, sf);  r[3] = sf;                              // scalar DFMA warp instructions per clock and SM, 4 scalar warps alone
    mix(16, 4, dm, sf); r[4] = sf; r[5] = dm;                   // the same 4 scalar warps next to 16 DMMA warps, and what the DMMA warps got
    e = cudaDeviceSynchronize();
    count_launch(6);
    cudaFree(d_out); cudaFree(d_cnt);
    if (e != cudaSuccess) return fail_cuda(e, "probe_fp64_pipe");
    return E2E_OK;
}

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
