// qmc_det_kinetic: the determinant's kinetic term of the local energy (eq. 3 first term,
// eq. 37; L401 "collected after all Monte Carlo walkers have advanced one step").  For Psi = det A
// only row i of A depends on r_i, so (cofactor expansion along row i, B = (A^-1)^T)
//     grad_i det A / det A = sum_j grad phi_j(r_i) B[i][j],   lap_i det A / det A = sum_j lap phi_j(r_i) B[i][j]
// and sum_j phi_j(r_i) B[i][j] = 1 checks that B is the inverse at these positions.  The SPO-VGL of
// the electrons' CURRENT positions comes from the same batched gather kernel the sweep uses, spo_batch
// electrons of every walker per launch; this consumes value, gradient and Laplacian of S2.
#include <mutex>

#include "delayed_device.cuh"

namespace qmc {

// One block per (electron of the chunk, walker): five fp64 dots of row iel0 + j of B with the fp32
// vectors v, d/dx, d/dy, d/dz, lap of that electron (fixed order: bit-reproducible).
template <typename TB>
__global__ void __launch_bounds__(256)
det_glap_kernel(const TB *__restrict__ B, int nel, int ld, int np, int nw, int iel0,
                const float *__restrict__ vgl, double *__restrict__ grad_out, double *__restrict__ lap_out,
                double *__restrict__ one_out)
{
    __shared__ double red[33];
    const int j = blockIdx.x, w = blockIdx.y, i = iel0 + j;
    const TB *row = B + ((size_t)w * nel + i) * ld;
    const float *x = vgl + ((size_t)j * nw + w) * 5 * np;
    double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    for (int c = threadIdx.x; 2 * c < nel; c += 256) {      // the vectors are zero-padded up to np >= nel
        const double2 b = ld2(row + 2 * c);
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const float2 f = reinterpret_cast<const float2 *>(x + (size_t)k * np)[c];
            acc[k] = fma(b.x, (double)f.x, acc[k]);
            acc[k] = fma(b.y, (double)f.y, acc[k]);
        }
    }
#pragma unroll
    for (int k = 0; k < 5; ++k) acc[k] = block_sum(acc[k], red);
    if (threadIdx.x == 0) {
        const size_t e = (size_t)w * nel + i;
        if (one_out) one_out[e] = acc[0];
        if (grad_out) { grad_out[3 * e + 0] = acc[1]; grad_out[3 * e + 1] = acc[2]; grad_out[3 * e + 2] = acc[3]; }
        lap_out[e] = acc[4];
    }
}

// ekin[w] = -1/2 sum_i lap[w][i]; one block per walker, fixed order.
__global__ void __launch_bounds__(256) ekin_kernel(const double *__restrict__ lap, int nel, double *__restrict__ ekin)
{
    __shared__ double red[33];
    const int w = blockIdx.x;
    double acc = 0.0;
    for (int i = threadIdx.x; i < nel; i += 256) acc += lap[(size_t)w * nel + i];
    acc = block_sum(acc, red);
    if (threadIdx.x == 0) ekin[w] = -0.5 * acc;
}

}  // namespace qmc

using namespace qmc;

extern "C" int qmc_det_kinetic(qmc_det_t *d, const qmc_spline_t *sp, const double *pos, double *grad_out,
                               double *lap_out, double *one_out, double *ekin_out, void *stream)
{
    QMC_REQUIRE(d && sp && pos, "qmc_det_kinetic: NULL argument");
    QMC_REQUIRE(d->spline == sp, "qmc_det_kinetic: the determinant was initialised from another spline");
    QMC_REQUIRE(grad_out || lap_out || one_out || ekin_out, "qmc_det_kinetic: no output requested");
    cudaStream_t s = (cudaStream_t)stream;
    if (d->delay) {               // the inverse must be current
        int rc = delayed_flush_reset_host(d, s);
        if (rc) return rc;
    }
    double *lap = lap_out;
    if (!lap) {
        if (!d->kin_lap) {
            cudaError_t e = cudaMalloc((void **)&d->kin_lap, (size_t)d->nw * d->nel * sizeof(double));
            if (e != cudaSuccess) {
                set_error("qmc_det_kinetic: cudaMalloc -> %s", cudaGetErrorString(e));
                (void)cudaGetLastError();
                return QMC_ENOMEM;
            }
        }
        lap = d->kin_lap;
    }
    for (int k = 0; k < d->nel; k += d->spo_batch) {
        const int nb = d->nel - k < d->spo_batch ? d->nel - k : d->spo_batch;
        int rc = spo_batch_vgl(d, sp, pos, nullptr, k, nb, nullptr, 0, d->vgl, s);
        if (rc) return rc;
        QMC_WITH_B(d, TB, Bp, (det_glap_kernel<TB><<<dim3(nb, d->nw), 256, 0, s>>>(Bp, d->nel, d->ld, d->np, d->nw, k, d->vgl, grad_out, lap, one_out)));
        QMC_LAUNCHED();
    }
    if (ekin_out) {
        ekin_kernel<<<d->nw, 256, 0, s>>>(lap, d->nel, ekin_out);
        QMC_LAUNCHED();
    }
    return QMC_OK;
}

// ---------------------------------------------------------------------------------------------------
// qmc_det_kinetic_noalloc: E_kin per walker with the per-electron Laplacians staged in a file-scope device
// array instead of a buffer from cudaMalloc (callers that may not allocate: include/qmc_b200.h).  Same
// kernels, same launch shapes and same summation order as qmc_det_kinetic(..., ekin_out): the same bits.
//
// The array is part of the library image: every GPU that loads the library holds its 4 MiB until exit.
// Every call on a device uses the same array; nothing in it has to start at zero (det_glap_kernel
// overwrites the nw * nel elements ekin_kernel reads, on the same stream, before they are read), and what a
// call leaves behind is never read by the next.  Calls that overlap on the GPU (two streams, two host
// threads) race on it.
static_assert(QMC_KINETIC_NOALLOC_MAX == (1 << 19), "the header states the limit in elements and bytes");
static __device__ __align__(256) double g_kin_lap_static[QMC_KINETIC_NOALLOC_MAX];

// Device address of g_kin_lap_static on `device`, which must be the current one.  In host code the array's
// name is only the symbol's host-side stand-in; the address a kernel can use comes from the runtime, once
// per device.
static int kin_static_scratch(int device, double **out)
{
    constexpr int kMaxDevices = 64;
    static double *ptr[kMaxDevices] = {};
    static std::mutex mu;
    int cur = -1;
    QMC_CUDA(cudaGetDevice(&cur));
    QMC_REQUIRE(cur == device, "qmc_det_kinetic_noalloc: the handle lives on device %d, the current device is %d", device, cur);
    QMC_REQUIRE(device >= 0 && device < kMaxDevices, "qmc_det_kinetic_noalloc: device ordinal %d not supported", device);
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[device]) {
        double *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void **)&p, g_kin_lap_static);
        if (e != cudaSuccess || !p) {
            set_error("qmc_det_kinetic_noalloc: cudaGetSymbolAddress -> %s", cudaGetErrorString(e));
            (void)cudaGetLastError();
            return QMC_ECUDA;
        }
        ptr[device] = p;
    }
    *out = ptr[device];
    return QMC_OK;
}

extern "C" int qmc_det_kinetic_noalloc(qmc_det_t *d, const qmc_spline_t *sp, const double *pos, double *ekin_out,
                                       void *stream)
{
    QMC_REQUIRE(d && sp && pos && ekin_out, "qmc_det_kinetic_noalloc: NULL argument");
    QMC_REQUIRE(d->spline == sp, "qmc_det_kinetic_noalloc: the determinant was initialised from another spline");
    const size_t need = (size_t)d->nw * d->nel;
    QMC_REQUIRE(need <= (size_t)QMC_KINETIC_NOALLOC_MAX,
                "qmc_det_kinetic_noalloc: nwalkers * nel = %zu exceeds the static scratch of %d elements "
                "(QMC_KINETIC_NOALLOC_MAX); use qmc_det_kinetic", need, (int)QMC_KINETIC_NOALLOC_MAX);
    double *lap = nullptr;
    int rc = kin_static_scratch(d->device, &lap);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    if (d->delay) {               // the inverse must be current
        rc = delayed_flush_reset_host(d, s);
        if (rc) return rc;
    }
    for (int k = 0; k < d->nel; k += d->spo_batch) {
        const int nb = d->nel - k < d->spo_batch ? d->nel - k : d->spo_batch;
        rc = spo_batch_vgl(d, sp, pos, nullptr, k, nb, nullptr, 0, d->vgl, s);
        if (rc) return rc;
        QMC_WITH_B(d, TB, Bp, (det_glap_kernel<TB><<<dim3(nb, d->nw), 256, 0, s>>>(Bp, d->nel, d->ld, d->np, d->nw, k, d->vgl, nullptr, lap, nullptr)));
        QMC_LAUNCHED();
    }
    ekin_kernel<<<d->nw, 256, 0, s>>>(lap, d->nel, ekin_out);
    QMC_LAUNCHED();
    return QMC_OK;
}
