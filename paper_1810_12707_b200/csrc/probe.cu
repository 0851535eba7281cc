// probe.cu — measurement helpers behind mhd_probe_*: not part of the method, used by bench.py for the roofline denominators.
//
// fp64 issue peak: SURVEY.md §8(d) asks for an FMA micro-benchmark because MEASURED_PEAKS.json holds no fp64 figure.
// Every thread runs 16 independent DFMA chains (no memory traffic); 8 CTAs of 256 threads per SM keep all four
// schedulers' fp64 pipes saturated.  The result is fp64 instructions per second (a DADD / DMUL occupies the same issue
// slot as a DFMA, so this is the ceiling of the butterfly-heavy fused x sweep); flop/s = 2 x that for pure FMA code.
#include "ctx.h"

namespace {

__global__ void __launch_bounds__(256) fp64_fma_kernel(double* out, int iters, double a, double b) {
    double x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = (double)(threadIdx.x + i) * 1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, b);
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == 123.456) out[0] = s;       // never true: keeps the chains alive
}

}  // namespace

extern "C" int mhd_probe_fp64(mhd_ctx* c, double* instr_per_s) {
    if (!c || !instr_per_s) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = sms * 8, threads = 256, iters = 4096;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, c->st);
        fp64_fma_kernel<<<blocks, threads, 0, c->st>>>(c->res, iters, 0.999999, 1e-9);
        cudaEventRecord(e1, c->st);
        cudaEventSynchronize(e1);
        float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
        const double n = (double)blocks * threads * iters * 64.0;
        if (rep > 0 && ms > 0) best = std::max(best, n / (ms * 1e-3));
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    c->launches += 4;
    *instr_per_s = best;
    return check_cuda(c, "probe_fp64");
}
