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

// qmc_probe_fp64_pipe: how the fp64 pipe of an SM sub-partition behaves -- the facts the flush kernels are laid
// out around (profiles/r02_fp64_pipe.md).  MODE 0: DMMA only; 1: DFMA only; 2: one DMMA + two DFMA per slot.
// NC independent accumulator chains per warp, `warps` warps per SM (one CTA per SM).
template <int NC, int MODE>
__global__ void __launch_bounds__(1024) fp64_pipe_kernel(double *out, int iters, double a0, double b0)
{
    double c[NC][2], f[NC][2];
#pragma unroll
    for (int i = 0; i < NC; ++i) { c[i][0] = c[i][1] = 0.0; f[i][0] = f[i][1] = 1.0; }
    const double a = a0 + threadIdx.x, b = b0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            if (MODE != 1)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
            if (MODE != 0) {
                asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(f[i][0]) : "d"(a), "d"(b));
                asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(f[i][1]) : "d"(a), "d"(b));
            }
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) s += c[i][0] + c[i][1] + f[i][0] + f[i][1];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace qmc

using namespace qmc;

extern "C" int qmc_probe_fp64_pipe(int mode, int warps_per_sm, int chains, double *tflops_dmma_host,
                                   double *tflops_dfma_host, void *stream)
{
    QMC_REQUIRE(tflops_dmma_host && tflops_dfma_host, "qmc_probe_fp64_pipe: NULL argument");
    QMC_REQUIRE(mode >= 0 && mode <= 2 && warps_per_sm >= 1 && warps_per_sm <= 32 && (chains == 1 || chains == 2 || chains == 4 || chains == 8),
                "qmc_probe_fp64_pipe: mode=%d warps_per_sm=%d chains=%d", mode, warps_per_sm, chains);
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, nsm = 0;
    QMC_CUDA(cudaGetDevice(&dev));
    QMC_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    double *out = nullptr;
    QMC_CUDA(cudaMalloc(&out, (size_t)nsm * 1024 * sizeof(double)));
    cudaEvent_t e0, e1;
    QMC_CUDA(cudaEventCreate(&e0));
    QMC_CUDA(cudaEventCreate(&e1));
    const int iters = 4096;
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, s);
#define QMC_PIPE(NC, M) fp64_pipe_kernel<NC, M><<<nsm, 32 * warps_per_sm, 0, s>>>(out, iters, 1.0, 1.0)
#define QMC_PIPE_NC(M) do { if (chains == 1) QMC_PIPE(1, M); else if (chains == 2) QMC_PIPE(2, M); else if (chains == 4) QMC_PIPE(4, M); else QMC_PIPE(8, M); } while (0)
        if (mode == 0) QMC_PIPE_NC(0); else if (mode == 1) QMC_PIPE_NC(1); else QMC_PIPE_NC(2);
#undef QMC_PIPE_NC
#undef QMC_PIPE
        cudaEventRecord(e1, s);
        count_launch();
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(out); set_error("qmc_probe_fp64_pipe: %s", cudaGetErrorString(e)); return QMC_ECUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep >= 1 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    const double slots = (double)nsm * warps_per_sm * iters * chains;     // warp-level slots executed
    *tflops_dmma_host = mode != 1 ? slots * 512.0 / (best * 1e-3) / 1e12 : 0.0;            // 8x8x4 MACs = 512 flop
    *tflops_dfma_host = mode != 0 ? slots * 2.0 * 64.0 / (best * 1e-3) / 1e12 : 0.0;      // two warp-wide FMAs = 128 flop
    return QMC_OK;
}

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
