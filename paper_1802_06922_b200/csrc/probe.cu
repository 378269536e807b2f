// qmc_probe_fp64_dmma: measured peak of the fp64 tensor-core path (mma.sync.m8n8k4.f64, SASS
// DMMA.8x8x4) on this device -- the denominator bench.py uses for the flush kernel's tensor-pipe
// utilisation (MEASURED_PEAKS.json has no fp64 figure).  An issue loop with independent
// accumulators and register operands, one CTA of 16 warps per SM: nothing but the tensor pipe.
#include "dmma.cuh"

namespace qmc {

constexpr int kProbeAcc = 8;

__global__ void __launch_bounds__(512) dmma_probe_kernel(double *out, int iters, double a0, double b0)
{
    double c[kProbeAcc][2];
#pragma unroll
    for (int i = 0; i < kProbeAcc; ++i) c[i][0] = c[i][1] = 0.0;
    const double a = a0 + threadIdx.x, b = b0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < kProbeAcc; ++i) {
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1])
                         : "d"(a), "d"(b));
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kProbeAcc; ++i) s += c[i][0] + c[i][1];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace qmc

using namespace qmc;

extern "C" int qmc_probe_fp64_dmma(double *tflops_host, void *stream)
{
    QMC_REQUIRE(tflops_host, "qmc_probe_fp64_dmma: NULL argument");
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, nsm = 0;
    QMC_CUDA(cudaGetDevice(&dev));
    QMC_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    double *out = nullptr;
    QMC_CUDA(cudaMalloc(&out, (size_t)nsm * 512 * sizeof(double)));
    cudaEvent_t e0, e1;
    QMC_CUDA(cudaEventCreate(&e0));
    QMC_CUDA(cudaEventCreate(&e1));
    const int iters = 8192;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {      // the first repetitions warm the clocks up
        cudaEventRecord(e0, s);
        dmma_probe_kernel<<<nsm, 512, 0, s>>>(out, iters, 1.0, 1.0);
        cudaEventRecord(e1, s);
        count_launch();
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(out); set_error("qmc_probe_fp64_dmma: %s", cudaGetErrorString(e)); return QMC_ECUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = (double)nsm * 16 * iters * kProbeAcc * 512.0;   // 8x8x4 MACs = 512 flop per warp instruction
        const double tf = flops / (ms * 1e-3) / 1e12;
        if (rep >= 1 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    *tflops_host = best;
    return QMC_OK;
}
