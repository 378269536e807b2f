// qmc_spline_* and qmc_spo_vgl: the fp32 orbital-innermost coefficient table and the SPO-VGL
// gather (sec 6.2.1).  See include/qmc_b200.h for the contract.
#include <math.h>

#include <atomic>
#include <string>

#include "spo_device.cuh"

namespace qmc {

static thread_local std::string g_err;
static std::atomic<long long> g_launches{0};

void set_error(const char *fmt, ...)
{
    char buf[1024];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
}
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

static bool invert3(const double *L, double *Li)
{
    const double c00 = L[4] * L[8] - L[5] * L[7];
    const double c01 = L[5] * L[6] - L[3] * L[8];
    const double c02 = L[3] * L[7] - L[4] * L[6];
    const double det = L[0] * c00 + L[1] * c01 + L[2] * c02;
    if (det == 0.0 || !isfinite(det)) return false;
    const double id = 1.0 / det;
    Li[0] = c00 * id;
    Li[1] = (L[2] * L[7] - L[1] * L[8]) * id;
    Li[2] = (L[1] * L[5] - L[2] * L[4]) * id;
    Li[3] = c01 * id;
    Li[4] = (L[0] * L[8] - L[2] * L[6]) * id;
    Li[5] = (L[2] * L[3] - L[0] * L[5]) * id;
    Li[6] = c02 * id;
    Li[7] = (L[1] * L[6] - L[0] * L[7]) * id;
    Li[8] = (L[0] * L[4] - L[1] * L[3]) * id;
    return true;
}

// One block per (orbital tile, position); each thread owns four consecutive orbitals and walks
// the 64 stencil rows with 128-bit streaming loads (rows are 128-byte aligned, so a warp reads
// 512 contiguous bytes per row).
template <bool WITH_GL>
__global__ void __launch_bounds__(256)
spo_vgl_kernel(SplineView sp, int npos, const double *__restrict__ pos, float *__restrict__ v,
               float *__restrict__ g, float *__restrict__ l, int ldo)
{
    __shared__ StencilSmem st;
    const int p = blockIdx.y;
    stage_stencil(sp, pos[3 * (size_t)p + 0], pos[3 * (size_t)p + 1], pos[3 * (size_t)p + 2], st);
    const int col = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
    if (col >= sp.np) return;
    float4 fv, gx, gy, gz, lp;
    gather4<WITH_GL>(sp, st, col, fv, gx, gy, gz, lp);
    if (col < ldo) {
        *reinterpret_cast<float4 *>(v + (size_t)p * ldo + col) = fv;
        if (WITH_GL) {
            float *gp = g + (size_t)p * 3 * ldo + col;
            *reinterpret_cast<float4 *>(gp) = gx;
            *reinterpret_cast<float4 *>(gp + ldo) = gy;
            *reinterpret_cast<float4 *>(gp + 2 * (size_t)ldo) = gz;
            *reinterpret_cast<float4 *>(l + (size_t)p * ldo + col) = lp;
        }
    }
}

// Threads per block / tiles for a row pitch np (multiple of 32 floats).
void spo_launch_shape(int np, int *threads, int *tiles)
{
    const int quads = np / 4;              // multiple of 8
    int t = quads < 256 ? quads : 256;
    t = (t + 31) / 32 * 32;
    *threads = t;
    *tiles = (quads + t - 1) / t;
}

}  // namespace qmc

using namespace qmc;

extern "C" const char *qmc_last_error(void) { return g_err.c_str(); }
extern "C" long long qmc_launch_count(void) { return g_launches.load(); }

extern "C" int qmc_spline_create(qmc_spline_t **out, int nx, int ny, int nz, int norb,
                                 const double *lattice, const float *coefs, int coefs_on_device,
                                 void *stream)
{
    QMC_REQUIRE(out && lattice && coefs, "qmc_spline_create: NULL argument");
    *out = nullptr;
    QMC_REQUIRE(nx >= 1 && ny >= 1 && nz >= 1 && norb >= 1,
                "qmc_spline_create: bad sizes nx=%d ny=%d nz=%d norb=%d", nx, ny, nz, norb);
    double li[9];
    QMC_REQUIRE(invert3(lattice, li), "qmc_spline_create: lattice is singular");
    cudaStream_t s = (cudaStream_t)stream;
    qmc_spline *h = new (std::nothrow) qmc_spline();
    if (!h) { set_error("qmc_spline_create: host allocation failed"); return QMC_ENOMEM; }
    SplineView &sv = h->view;
    sv.nx = nx; sv.ny = ny; sv.nz = nz; sv.norb = norb;
    sv.np = (norb + 31) / 32 * 32;
    const int nd[3] = {nx, ny, nz};
    for (int j = 0; j < 3; ++j)
        for (int d = 0; d < 3; ++d) {
            sv.linv[3 * j + d] = li[3 * j + d];
            sv.jac[3 * j + d] = li[3 * j + d] * (double)nd[d];
        }
    const int de[6][2] = {{0, 0}, {1, 1}, {2, 2}, {0, 1}, {0, 2}, {1, 2}};
    for (int q = 0; q < 6; ++q) {
        double acc = 0.0;
        for (int j = 0; j < 3; ++j) acc += sv.jac[3 * j + de[q][0]] * sv.jac[3 * j + de[q][1]];
        sv.metric[q] = acc;
    }
    const size_t rows = (size_t)nx * ny * nz;
    h->bytes = rows * sv.np * sizeof(float);
    cudaError_t e = cudaMalloc(&h->coefs, h->bytes);
    if (e != cudaSuccess) {
        set_error("qmc_spline_create: cudaMalloc(%zu bytes) -> %s", h->bytes, cudaGetErrorString(e));
        delete h;
        (void)cudaGetLastError();
        return QMC_ENOMEM;
    }
    sv.coefs = h->coefs;
    const cudaMemcpyKind kind = coefs_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    if (sv.np == norb) {
        e = cudaMemcpyAsync(h->coefs, coefs, h->bytes, kind, s);
    } else {
        e = cudaMemsetAsync(h->coefs, 0, h->bytes, s);
        if (e == cudaSuccess)
            e = cudaMemcpy2DAsync(h->coefs, (size_t)sv.np * sizeof(float), coefs,
                                  (size_t)norb * sizeof(float), (size_t)norb * sizeof(float), rows,
                                  kind, s);
    }
    if (e != cudaSuccess) {
        set_error("qmc_spline_create: table copy -> %s", cudaGetErrorString(e));
        cudaFree(h->coefs);
        delete h;
        return QMC_ECUDA;
    }
    *out = h;
    return QMC_OK;
}

extern "C" int qmc_spline_destroy(qmc_spline_t *h)
{
    if (!h) return QMC_OK;
    cudaError_t e = cudaFree(h->coefs);
    delete h;
    if (e != cudaSuccess) { set_error("qmc_spline_destroy: %s", cudaGetErrorString(e)); return QMC_ECUDA; }
    return QMC_OK;
}

extern "C" int qmc_spline_set_half_twist(qmc_spline_t *h, const int *half_twist)
{
    QMC_REQUIRE(h && half_twist, "qmc_spline_set_half_twist: NULL argument");
    for (int d = 0; d < 3; ++d)
        QMC_REQUIRE(half_twist[d] == 0 || half_twist[d] == 1,
                    "qmc_spline_set_half_twist: half_twist[%d]=%d is neither 0 nor 1", d, half_twist[d]);
    for (int d = 0; d < 3; ++d) h->view.half_twist[d] = half_twist[d];
    return QMC_OK;
}

extern "C" int qmc_spline_info(const qmc_spline_t *h, int *row_pitch, size_t *table_bytes)
{
    QMC_REQUIRE(h, "qmc_spline_info: NULL handle");
    if (row_pitch) *row_pitch = h->view.np;
    if (table_bytes) *table_bytes = h->bytes;
    return QMC_OK;
}

extern "C" int qmc_spo_vgl(const qmc_spline_t *h, int npos, const double *pos, float *v, float *g,
                           float *l, int ldo, void *stream)
{
    QMC_REQUIRE(h, "qmc_spo_vgl: NULL spline");
    QMC_REQUIRE(npos >= 0, "qmc_spo_vgl: npos=%d", npos);
    if (npos == 0) return QMC_OK;
    QMC_REQUIRE(pos && v, "qmc_spo_vgl: NULL pos or v");
    QMC_REQUIRE((g == nullptr) == (l == nullptr), "qmc_spo_vgl: g and l must be given together");
    QMC_REQUIRE(ldo >= h->view.norb && ldo % 4 == 0, "qmc_spo_vgl: ldo=%d must be >= norb=%d and a multiple of 4",
                ldo, h->view.norb);
    QMC_REQUIRE(((uintptr_t)v % 16 == 0) && ((uintptr_t)g % 16 == 0) && ((uintptr_t)l % 16 == 0),
                "qmc_spo_vgl: outputs must be 16-byte aligned");
    int threads, tiles;
    spo_launch_shape(h->view.np, &threads, &tiles);
    cudaStream_t s = (cudaStream_t)stream;
    // grid.y is limited to 65535 blocks
    for (int p0 = 0; p0 < npos; p0 += 65535) {
        const int n = npos - p0 < 65535 ? npos - p0 : 65535;
        dim3 grid(tiles, n);
        const double *pp = pos + 3 * (size_t)p0;
        float *vp = v + (size_t)p0 * ldo;
        if (g) {
            spo_vgl_kernel<true><<<grid, threads, 0, s>>>(h->view, n, pp, vp, g + (size_t)p0 * 3 * ldo,
                                                          l + (size_t)p0 * ldo, ldo);
        } else {
            spo_vgl_kernel<false><<<grid, threads, 0, s>>>(h->view, n, pp, vp, nullptr, nullptr, ldo);
        }
        QMC_LAUNCHED();
    }
    return QMC_OK;
}
