// nk_probe.cu -- the fp64 ceiling of this GPU, measured: a DFMA-only microbenchmark ("no fp64
// peak measured yet -- measure a DFMA microbenchmark"; BASELINE.json north_star asks for fp64-pipe evidence
// beside the HBM roofline).  ax_e's arithmetic intensity (1.7 - 3.2 flop/B at N = 7..15) sits below the
// machine balance, so HBM bounds it; this number is the SECONDARY roofline its executed DFMA rate is quoted
// against (bench.py "fp64").  Not on the hot path.
#include "nk_host.h"

namespace {

// Every thread runs CHAINS independent dependent-FMA chains (fp64 latency is hidden by the chains of one
// thread plus the other resident warps); operands live in registers; the result is stored so that nothing
// is optimised away.  2 flops per DFMA.
constexpr int CHAINS = 8;
constexpr int THREADS = 256;

__global__ void __launch_bounds__(THREADS)
dfma_probe_kernel(double *sink, int iters, double a, double b)
{
    double acc[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) acc[c] = (double)(threadIdx.x + c);
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int c = 0; c < CHAINS; ++c) acc[c] = fma(acc[c], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += acc[c];
    if (s == 123.456) sink[0] = s;        // never true for a = 1 - 2^-30, b = 2^-30 and finite iteration counts
}

}  // namespace

extern "C" int nk_fp64_peak(double *tflops_host, double *dfma_per_clk_per_sm_host, void *stream)
{
    if (!tflops_host) return NK_ERR_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int dev = 0, sms = 0, khz = 0;
    NK_CUDA(cudaGetDevice(&dev));
    NK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    NK_CUDA(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
    double *sink = nullptr;
    NK_CUDA(cudaMalloc(&sink, sizeof(double)));
    cudaEvent_t e0, e1;
    NK_CUDA(cudaEventCreate(&e0));
    NK_CUDA(cudaEventCreate(&e1));
    const int blocks = sms * 8;            // 8 resident CTAs of 256 threads per SM = 64 warps: full occupancy
    const int iters = 4096;
    const double a = 1.0 - 1.0 / 1073741824.0, b = 1.0 / 1073741824.0;
    double best_ms = 1e30;
    cudaError_t e = cudaSuccess;
    for (int rep = 0; rep < 6 && e == cudaSuccess; ++rep) {     // first repetition warms the clocks up
        cudaEventRecord(e0, st);
        dfma_probe_kernel<<<blocks, THREADS, 0, st>>>(sink, iters, a, b);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (e != cudaSuccess) return nk_cuda_fail(e);
    const double dfma = (double)blocks * THREADS * (double)iters * 8.0 * CHAINS;
    *tflops_host = 2.0 * dfma / (best_ms * 1e-3) / 1e12;
    // against the device's maximum SM clock (the clock under this load is lower when the power cap bites)
    if (dfma_per_clk_per_sm_host) *dfma_per_clk_per_sm_host = dfma / (best_ms * 1e-3) / ((double)khz * 1e3) / sms;
    return NK_OK;
}
