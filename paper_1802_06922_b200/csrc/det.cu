// qmc_det_*: per-walker fp64 inverse of the Slater matrix, determinant ratio and
// Sherman-Morrison update (L299).  See include/qmc_b200.h for the contract.
#include <math.h>
#include <stdlib.h>

#include <new>
#include <vector>

#include "delayed_device.cuh"
#include "update_device.cuh"

namespace qmc {

// ---------------------------------------------------------------------------------------------
// det_init kernels

__global__ void init_stats_kernel(int nw, double *logdet, int *sign, long long *naccept)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < nw) { logdet[w] = 0.0; sign[w] = 1; if (naccept) naccept[w] = 0; }
}

// fp64 work matrix -> fp32 storage (one rounding to nearest even per element; R:A19), and dense
// [nw][nel][nel] double <-> padded [nw][nel][ld] TB for qmc_det_get_inverse / qmc_det_set_inverse.
__global__ void round_to_storage_kernel(const double *__restrict__ src, float *__restrict__ dst, size_t n)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        dst[i] = (float)src[i];
}
template <typename TB, bool UNPACK>
__global__ void pack_inverse_kernel(TB *__restrict__ B, double *__restrict__ dense, int nel, int ld)
{
    const size_t row = blockIdx.x;                       // w * nel + m
    TB *b = B + row * ld;
    double *o = dense + row * nel;
    for (int j = threadIdx.x; j < nel; j += blockDim.x) {
        if (UNPACK) o[j] = (double)b[j];
        else b[j] = (TB)o[j];
    }
}

// B[w][j][i] = (double) v[w][i][j]: the transposed Slater matrix, so that inverting it in place
// gives (A^T)^-1 = (A^-1)^T.  v is [nwc][nel][np] floats.  32x32 tiles through shared memory.
__global__ void fill_transposed_kernel(const float *__restrict__ v, int np, double *__restrict__ B,
                                       int nel, int ld)
{
    __shared__ float tile[32][33];
    const int w = blockIdx.z;
    const int i0 = blockIdx.y * 32, j0 = blockIdx.x * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int i = i0 + r, j = j0 + threadIdx.x;
        tile[r][threadIdx.x] = (i < nel && j < nel) ? v[((size_t)w * nel + i) * np + j] : 0.f;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int j = j0 + r, i = i0 + threadIdx.x;
        if (j < nel && i < nel) B[((size_t)w * nel + j) * ld + i] = (double)tile[threadIdx.x][r];
    }
}

// Gauss-Jordan step k, part 1 (one block per walker): partial pivot search in column k, scaled
// pivot row, old row k, the multiplier column (indexed after the row swap), log|det| and sign.
__global__ void __launch_bounds__(256)
gj_pivot_kernel(double *__restrict__ B, int nel, int ld, int k, int *__restrict__ piv,
                double *__restrict__ prow, double *__restrict__ krow, double *__restrict__ fcol,
                double *__restrict__ logdet, int *__restrict__ sign, int *__restrict__ singular)
{
    __shared__ double s_val[256];
    __shared__ int s_idx[256];
    const int w = blockIdx.x, tid = threadIdx.x;
    double *M = B + (size_t)w * nel * ld;
    double *fc = fcol + (size_t)w * nel;
    double best = -1.0;
    int bi = k;
    for (int i = tid; i < nel; i += 256) {
        const double c = M[(size_t)i * ld + k];
        fc[i] = c;
        const double ac = fabs(c);
        if (i >= k && (ac > best)) { best = ac; bi = i; }   // lowest index wins ties per thread
    }
    s_val[tid] = best;
    s_idx[tid] = bi;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (tid < s) {
            const double ov = s_val[tid + s];
            const int oi = s_idx[tid + s];
            if (ov > s_val[tid] || (ov == s_val[tid] && oi < s_idx[tid])) { s_val[tid] = ov; s_idx[tid] = oi; }
        }
        __syncthreads();
    }
    const int p = s_idx[0];
    const double d = M[(size_t)p * ld + k];
    const bool bad = !(fabs(d) > 0.0) || !isfinite(d);
    const double dinv = bad ? 1.0 : 1.0 / d;
    const double ckk = M[(size_t)k * ld + k];
    __syncthreads();
    if (tid == 0) {
        piv[(size_t)w * nel + k] = p;
        if (bad) singular[w] = 1;
        else {
            logdet[w] += log(fabs(d));
            if ((d < 0.0) != (p != k)) sign[w] = -sign[w];
        }
        fc[p] = ckk;      // after the swap row p holds the old row k
    }
    double *pr = prow + (size_t)w * ld, *kr = krow + (size_t)w * ld;
    for (int j = tid; j < ld; j += 256) {
        const double x = (j == k) ? 1.0 : M[(size_t)p * ld + j];
        pr[j] = x * dinv;
        kr[j] = M[(size_t)k * ld + j];
    }
}

// Gauss-Jordan step k, part 2: every row i != k becomes row_i (column k zeroed) - f_i * prow;
// row k becomes prow; row p takes the old row k.  Elementwise, 16 bytes/element of traffic.
constexpr int kGjRows = 8;
__global__ void __launch_bounds__(256)
gj_eliminate_kernel(double *__restrict__ B, int nel, int ld, int k, const int *__restrict__ piv,
                    const double *__restrict__ prow, const double *__restrict__ krow,
                    const double *__restrict__ fcol)
{
    const int w = blockIdx.y;
    const int p = piv[(size_t)w * nel + k];
    double *M = B + (size_t)w * nel * ld;
    const double2 *pr = reinterpret_cast<const double2 *>(prow + (size_t)w * ld);
    const double2 *kr = reinterpret_cast<const double2 *>(krow + (size_t)w * ld);
    const double *fc = fcol + (size_t)w * nel;
    const int i0 = blockIdx.x * kGjRows, i1 = min(nel, i0 + kGjRows);
    for (int c = threadIdx.x; c < ld / 2; c += 256) {
        const double2 pv = pr[c];
        const bool hasx = (2 * c == k), hasy = (2 * c + 1 == k);
        for (int i = i0; i < i1; ++i) {
            double2 *row = reinterpret_cast<double2 *>(M + (size_t)i * ld);
            double2 out;
            if (i == k) out = pv;
            else {
                double2 src = (i == p) ? kr[c] : row[c];
                if (hasx) src.x = 0.0;
                if (hasy) src.y = 0.0;
                const double f = fc[i];
                out.x = fma(-f, pv.x, src.x);
                out.y = fma(-f, pv.y, src.y);
            }
            row[c] = out;
        }
    }
}

// Net column order after undoing the row interchanges: out[:, j] = M[:, idx[j]].
__global__ void gj_perm_kernel(int nw, int nel, const int *__restrict__ piv, int *__restrict__ idx)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= nw) return;
    int *ix = idx + (size_t)w * nel;
    const int *pv = piv + (size_t)w * nel;
    for (int j = 0; j < nel; ++j) ix[j] = j;
    for (int k = nel - 1; k >= 0; --k) {
        const int p = pv[k];
        const int t = ix[k]; ix[k] = ix[p]; ix[p] = t;
    }
}

__global__ void __launch_bounds__(256)
gj_unscramble_kernel(double *__restrict__ B, int nel, int ld, const int *__restrict__ idx)
{
    extern __shared__ double s_row[];
    const int w = blockIdx.y, i = blockIdx.x;
    double *row = B + ((size_t)w * nel + i) * ld;
    const int *ix = idx + (size_t)w * nel;
    for (int j = threadIdx.x; j < nel; j += 256) s_row[j] = row[j];
    __syncthreads();
    for (int j = threadIdx.x; j < nel; j += 256) row[j] = s_row[ix[j]];
}

// ---------------------------------------------------------------------------------------------
// ratio and row copy

// R_w = sum_j B_w[iel][j] * (double)phi_w[j]; one block per walker, fixed summation order.
template <typename TB>
__global__ void __launch_bounds__(128)
ratio_kernel(const TB *__restrict__ B, int nel, int ld, int iel, const float *__restrict__ phi,
             int ldphi, double *__restrict__ ratio)
{
    __shared__ double red[33];
    const int w = blockIdx.x;
    const TB *row = B + ((size_t)w * nel + iel) * ld;
    const float *ph = phi + (size_t)w * ldphi;
    double acc = 0.0;
    for (int j = threadIdx.x; j < nel; j += 128) acc = fma((double)row[j], (double)ph[j], acc);
    acc = block_sum(acc, red);
    if (threadIdx.x == 0) ratio[w] = acc;
}

// R[w][q] = sum_j B_w[iel][j] * (double)phi[w][q][j] for npts trial positions of the same electron: one
// block per walker, one warp per point (the row stays in L1/L2), fixed summation order per point.
template <typename TB>
__global__ void __launch_bounds__(256)
ratio_points_kernel(const TB *__restrict__ B, int nel, int ld, int iel, const float *__restrict__ phi,
                    int npts, int ldphi, double *__restrict__ ratios)
{
    const int w = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const TB *row = B + ((size_t)w * nel + iel) * ld;
    for (int q = warp; q < npts; q += 8) {
        const float *ph = phi + ((size_t)w * npts + q) * ldphi;
        double acc = 0.0;
        for (int j = lane; j < nel; j += 32) acc = fma((double)row[j], (double)ph[j], acc);
        acc = warp_sum(acc);
        if (lane == 0) ratios[(size_t)w * npts + q] = acc;
    }
}

template <typename TB>
__global__ void __launch_bounds__(256)
copy_rowk_kernel(const TB *__restrict__ B, int nel, int ld, int iel,
                 const unsigned char *__restrict__ accept, double *__restrict__ rowk)
{
    const int w = blockIdx.x;
    if (!accept[w]) return;
    const TB *row = B + ((size_t)w * nel + iel) * ld;
    double *dst = rowk + (size_t)w * ld;
    for (int j = threadIdx.x; j < ld; j += 256) dst[j] = (double)row[j];
}

template <typename T>
static int dev_alloc(T **p, size_t count, const char *what)
{
    *p = nullptr;
    if (count == 0) count = 1;
    cudaError_t e = cudaMalloc((void **)p, count * sizeof(T));
    if (e != cudaSuccess) {
        set_error("qmc_det: cudaMalloc(%s, %zu bytes) -> %s", what, count * sizeof(T), cudaGetErrorString(e));
        (void)cudaGetLastError();
        return QMC_ENOMEM;
    }
    return QMC_OK;
}

void prof_start(qmc_det *d, int kind, cudaStream_t s)
{
    if (!d->prof_on) return;
    if (!d->prof_events) { d->prof_events = new std::vector<cudaEvent_t>(); d->prof_kinds = new std::vector<int>(); }
    while (d->prof_events->size() < d->prof_used + 2) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) { d->prof_on = 0; return; }
        d->prof_events->push_back(e);
    }
    d->prof_kinds->resize(d->prof_used / 2 + 1);
    (*d->prof_kinds)[d->prof_used / 2] = kind;
    cudaEventRecord((*d->prof_events)[d->prof_used], s);
}

void prof_stop(qmc_det *d, cudaStream_t s)
{
    if (!d->prof_on) return;
    cudaEventRecord((*d->prof_events)[d->prof_used + 1], s);
    d->prof_used += 2;
}

static void det_free(qmc_det *d)
{
    if (!d) return;
    if (d->prof_events) {
        for (cudaEvent_t e : *d->prof_events) cudaEventDestroy(e);
        delete d->prof_events;
        delete d->prof_kinds;
    }
    if (d->aux) {
        cudaStreamSynchronize(d->aux);
        cudaEventDestroy(d->ev_spo[0]); cudaEventDestroy(d->ev_spo[1]); cudaEventDestroy(d->ev_main);
        cudaStreamDestroy(d->aux);
    }
    if (d->vgl_buf[1]) cudaFree(d->vgl_buf[1]);
    d->vgl = d->vgl_buf[0] ? d->vgl_buf[0] : d->vgl;
    cudaFree(d->cur); cudaFree(d->vgl_cur); cudaFree(d->rprop); cudaFree(d->fcur); cudaFree(d->tfac); cudaFree(d->jas_dj);
    cudaFree(d->B); cudaFree(d->Bf); cudaFree(d->logdet); cudaFree(d->sign); cudaFree(d->naccept);
    cudaFree(d->vgl); cudaFree(d->rowk); cudaFree(d->ratio); cudaFree(d->acc);
    cudaFree(d->win_count); cudaFree(d->win_iel); cudaFree(d->win_slot); cudaFree(d->win_phi); cudaFree(d->win_rows);
    cudaFree(d->win_sinv); cudaFree(d->win_full); cudaFree(d->stage); cudaFree(d->kin_lap);
    free(d->win_host_iel);
    delete d;
}

// In-place batched inverse of d->B (holding A^T) by Gauss-Jordan with partial pivoting.
static int invert_in_place(qmc_det *d, cudaStream_t s, bool *singular_out)
{
    const int nw = d->nw, nel = d->nel, ld = d->ld;
    int *piv = nullptr, *idx = nullptr, *sing = nullptr;
    double *prow = nullptr, *krow = nullptr, *fcol = nullptr;
    int rc = QMC_OK;
    auto cleanup = [&]() { cudaFree(piv); cudaFree(idx); cudaFree(sing); cudaFree(prow); cudaFree(krow); cudaFree(fcol); };
    if ((rc = dev_alloc(&piv, (size_t)nw * nel, "piv")) || (rc = dev_alloc(&idx, (size_t)nw * nel, "idx")) ||
        (rc = dev_alloc(&sing, (size_t)nw, "singular")) || (rc = dev_alloc(&prow, (size_t)nw * ld, "prow")) ||
        (rc = dev_alloc(&krow, (size_t)nw * ld, "krow")) || (rc = dev_alloc(&fcol, (size_t)nw * nel, "fcol"))) {
        cleanup();
        return rc;
    }
    cudaError_t e = cudaMemsetAsync(sing, 0, (size_t)nw * sizeof(int), s);
    for (int k = 0; k < nel && e == cudaSuccess; ++k) {
        gj_pivot_kernel<<<nw, 256, 0, s>>>(d->B, nel, ld, k, piv, prow, krow, fcol, d->logdet, d->sign, sing);
        dim3 grid((nel + kGjRows - 1) / kGjRows, nw);
        gj_eliminate_kernel<<<grid, 256, 0, s>>>(d->B, nel, ld, k, piv, prow, krow, fcol);
        count_launch(2);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        gj_perm_kernel<<<(nw + 63) / 64, 64, 0, s>>>(nw, nel, piv, idx);
        gj_unscramble_kernel<<<dim3(nel, nw), 256, (size_t)nel * sizeof(double), s>>>(d->B, nel, ld, idx);
        count_launch(2);
        e = cudaGetLastError();
    }
    std::vector<int> hs(nw, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(hs.data(), sing, (size_t)nw * sizeof(int), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cleanup();
    if (e != cudaSuccess) { set_error("qmc_det_init: inverse -> %s", cudaGetErrorString(e)); return QMC_ECUDA; }
    *singular_out = false;
    for (int w = 0; w < nw; ++w)
        if (hs[w]) { *singular_out = true; set_error("qmc_det_init: Slater matrix of walker %d is singular", w); break; }
    return QMC_OK;
}

// (A^-1)^T of every walker from the positions, into the handle's storage: Slater matrices by the
// SPO kernel (values only, in chunks of walkers), transposed into an fp64 work matrix, Gauss-Jordan in
// place, log|det| and sign from the pivots (logdet / sign must be 0 / +1 on entry).  With fp32
// storage the work matrix is temporary and rounded once into Bf.  Synchronises `s`.
static int build_inverse(qmc_det *d, const qmc_spline *sp, const double *pos, cudaStream_t s, bool *singular)
{
    const int nw = d->nw, nel = d->nel, ld = d->ld, np = d->np;
    const size_t nB = (size_t)nw * nel * ld;
    int rc;
    if (d->b32 && (rc = dev_alloc(&d->B, nB, "B (fp64 work matrix)"))) return rc;
    auto drop_work = [&]() { if (d->b32) { cudaFree(d->B); d->B = nullptr; } };
    cudaError_t e = cudaMemsetAsync(d->B, 0, nB * sizeof(double), s);
    if (e != cudaSuccess) { drop_work(); set_error("qmc_det: memset -> %s", cudaGetErrorString(e)); return QMC_ECUDA; }
    const size_t per_walker = (size_t)nel * np * sizeof(float);
    int wchunk = (int)((size_t)(256u << 20) / per_walker);
    if (wchunk < 1) wchunk = 1;
    if (wchunk > nw) wchunk = nw;
    float *vbuf = nullptr;
    if ((rc = dev_alloc(&vbuf, (size_t)wchunk * nel * np, "slater scratch"))) { drop_work(); return rc; }
    for (int w0 = 0; w0 < nw; w0 += wchunk) {
        const int nwc = nw - w0 < wchunk ? nw - w0 : wchunk;
        rc = qmc_spo_vgl(sp, nwc * nel, pos + (size_t)w0 * nel * 3, vbuf, nullptr, nullptr, np, s);
        if (rc) { cudaFree(vbuf); drop_work(); return rc; }
        dim3 grid((nel + 31) / 32, (nel + 31) / 32, nwc);
        fill_transposed_kernel<<<grid, dim3(32, 8), 0, s>>>(vbuf, np, d->B + (size_t)w0 * nel * ld, nel, ld);
        count_launch();
    }
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(vbuf);
    if (e != cudaSuccess) { drop_work(); set_error("qmc_det: Slater matrix -> %s", cudaGetErrorString(e)); return QMC_ECUDA; }
    rc = invert_in_place(d, s, singular);
    if (!rc && !*singular && d->b32) {
        round_to_storage_kernel<<<4 * d->nsm, 256, 0, s>>>(d->B, d->Bf, nB);
        count_launch();
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) { set_error("qmc_det: fp32 rounding -> %s", cudaGetErrorString(e)); rc = QMC_ECUDA; }
    }
    drop_work();
    return rc;
}

}  // namespace qmc

using namespace qmc;

extern "C" int qmc_det_init(qmc_det_t **out, const qmc_spline_t *sp, int nw, int nel, const double *pos,
                            int delay_rank, void *stream)
{
    return qmc_det_init_ex(out, sp, nw, nel, pos, delay_rank, 0, stream);
}

extern "C" int qmc_det_init_ex(qmc_det_t **out, const qmc_spline_t *sp, int nw, int nel, const double *pos,
                               int delay_rank, unsigned flags, void *stream)
{
    QMC_REQUIRE(out && sp && pos, "qmc_det_init: NULL argument");
    *out = nullptr;
    QMC_REQUIRE((flags & ~(unsigned)(QMC_DET_FP32_INVERSE | QMC_DET_ACCEPT_WINDOWS)) == 0, "qmc_det_init_ex: unknown flags 0x%x", flags);
    QMC_REQUIRE(!(flags & QMC_DET_ACCEPT_WINDOWS) || (delay_rank >= 2 && delay_rank <= 16),
                "qmc_det_init_ex: QMC_DET_ACCEPT_WINDOWS needs 2 <= delay_rank <= 16 (got %d)", delay_rank);
    QMC_REQUIRE(nw >= 1, "qmc_det_init: nwalkers=%d", nw);
    QMC_REQUIRE(nel == sp->view.norb, "qmc_det_init: nel=%d must equal the spline's norb=%d", nel, sp->view.norb);
    QMC_REQUIRE(nel <= kMaxNel, "qmc_det_init: nel=%d exceeds the supported maximum %d", nel, kMaxNel);
    QMC_REQUIRE(delay_rank >= 0 && delay_rank <= QMC_MAX_DELAY, "qmc_det_init: delay_rank=%d not in 0..%d",
                delay_rank, QMC_MAX_DELAY);
    QMC_REQUIRE(nw <= 65535, "qmc_det_init: nwalkers=%d exceeds 65535", nw);
    cudaStream_t s = (cudaStream_t)stream;
    qmc_det *d = new (std::nothrow) qmc_det();
    if (!d) { set_error("qmc_det_init: host allocation failed"); return QMC_ENOMEM; }
    d->spline = sp;
    QMC_CUDA_OR(cudaGetDevice(&d->device), det_free(d));
    QMC_CUDA_OR(cudaDeviceGetAttribute(&d->nsm, cudaDevAttrMultiProcessorCount, d->device), det_free(d));
    d->nw = nw; d->nel = nel; d->ld = update_ld(nel); d->np = sp->view.np;
    d->delay = delay_rank <= 1 ? 0 : delay_rank;
    d->spo_batch = d->delay ? d->delay : kSpoBatch;
    d->accept_windows = (flags & QMC_DET_ACCEPT_WINDOWS) ? 1 : 0;
    if (d->accept_windows) {
        d->spo_batch = d->delay + d->delay / 2;      // steps a window may take to collect `delay` accepts
        d->vgl_ring = 2 * d->spo_batch;
    }
    d->b32 = (flags & QMC_DET_FP32_INVERSE) ? 1 : 0;
    const int ld = d->ld, np = d->np, K = d->delay;
    int rc;
    if ((rc = d->b32 ? dev_alloc(&d->Bf, (size_t)nw * nel * ld, "B (fp32)") : dev_alloc(&d->B, (size_t)nw * nel * ld, "B")) ||
        (rc = dev_alloc(&d->logdet, nw, "logdet")) ||
        (rc = dev_alloc(&d->sign, nw, "sign")) || (rc = dev_alloc(&d->naccept, nw, "naccept")) ||
        (rc = dev_alloc(&d->vgl, (size_t)(d->accept_windows ? d->vgl_ring : d->spo_batch) * nw * 5 * np, "vgl")) ||
        (rc = dev_alloc(&d->rowk, (size_t)nw * ld, "rowk")) ||
        (rc = dev_alloc(&d->ratio, nw, "ratio")) ||
        (rc = dev_alloc(&d->acc, nw, "acc"))) {
        det_free(d);
        return rc;
    }
    d->vgl_buf[0] = d->vgl;
    if (K) {
        const char *env = getenv("QMC_SWEEP_OVERLAP");      // A/B measurements: 0 keeps everything on one stream
        d->overlap = !(env && atoi(env) == 0);
        if (d->overlap && !d->accept_windows && (rc = dev_alloc(&d->vgl_buf[1], (size_t)d->spo_batch * nw * 5 * np, "vgl (second buffer)"))) {
            det_free(d);
            return rc;
        }
    }
    if (K) {
        const int kmax = delayed_max_rank(ld);
        if (K > kmax) {
            set_error("qmc_det_init: delay_rank=%d does not fit shared memory for nel=%d (max %d)", K, nel, kmax);
            det_free(d);
            return QMC_EINVAL;
        }
        d->win_host_iel = (unsigned char *)calloc((size_t)nel, 1);
        if (!d->win_host_iel) { set_error("qmc_det_init: host allocation failed"); det_free(d); return QMC_ENOMEM; }
        if ((rc = dev_alloc(&d->win_count, nw, "win_count")) || (rc = dev_alloc(&d->win_iel, (size_t)nw * K, "win_iel")) ||
            (rc = dev_alloc(&d->win_slot, (size_t)nw * K, "win_slot")) ||
            (rc = dev_alloc(&d->win_phi, (size_t)nw * K * np, "win_phi")) ||
            (rc = dev_alloc(&d->win_rows, (size_t)nw * K * ld, "win_rows")) ||
            (rc = dev_alloc(&d->win_sinv, (size_t)nw * K * K, "win_sinv")) || (rc = dev_alloc(&d->win_full, 1, "win_full")) ||
            (d->accept_windows && (rc = dev_alloc(&d->cur, (size_t)2 * nw, "cur")))) {
            det_free(d);
            return rc;
        }
        d->win_vec = d->win_phi;
        d->win_vec_wstride = (size_t)K * np;
        d->win_vec_sstride = (size_t)np;
    }
    cudaError_t e = cudaMemsetAsync(d->rowk, 0, (size_t)nw * ld * sizeof(double), s);
    if (e == cudaSuccess) e = cudaMemsetAsync(d->vgl, 0, (size_t)(d->accept_windows ? d->vgl_ring : d->spo_batch) * nw * 5 * np * sizeof(float), s);
    if (e == cudaSuccess && d->vgl_buf[1]) e = cudaMemsetAsync(d->vgl_buf[1], 0, (size_t)d->spo_batch * nw * 5 * np * sizeof(float), s);
    if (e == cudaSuccess && K) e = cudaMemsetAsync(d->win_count, 0, (size_t)nw * sizeof(int), s);
    if (e == cudaSuccess && K) e = cudaMemsetAsync(d->win_full, 0, sizeof(int), s);
    if (e == cudaSuccess && K) e = cudaMemsetAsync(d->win_rows, 0, (size_t)nw * K * ld * sizeof(double), s);
    if (e != cudaSuccess) { set_error("qmc_det_init: memset -> %s", cudaGetErrorString(e)); det_free(d); return QMC_ECUDA; }
    init_stats_kernel<<<(nw + 127) / 128, 128, 0, s>>>(nw, d->logdet, d->sign, d->naccept);
    count_launch();
    bool singular = false;
    rc = build_inverse(d, sp, pos, s, &singular);
    if (rc) { det_free(d); return rc; }
    if (singular) { det_free(d); return QMC_ESINGULAR; }
    *out = d;
    return QMC_OK;
}

extern "C" int qmc_det_destroy(qmc_det_t *d)
{
    det_free(d);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("qmc_det_destroy: %s", cudaGetErrorString(e)); return QMC_ECUDA; }
    return QMC_OK;
}

extern "C" int qmc_det_profile(qmc_det_t *d, int enable)
{
    QMC_REQUIRE(d, "qmc_det_profile: NULL handle");
    d->prof_on = enable ? 1 : 0;
    d->prof_used = 0;
    return QMC_OK;
}

extern "C" int qmc_det_profile_read(qmc_det_t *d, double *ms, long long *launches)
{
    QMC_REQUIRE(d && ms && launches, "qmc_det_profile_read: NULL argument");
    for (int k = 0; k < kProfKinds; ++k) { ms[k] = 0.0; launches[k] = 0; }
    for (size_t i = 0; i + 1 < d->prof_used; i += 2) {
        QMC_CUDA(cudaEventSynchronize((*d->prof_events)[i + 1]));
        float t = 0.f;
        QMC_CUDA(cudaEventElapsedTime(&t, (*d->prof_events)[i], (*d->prof_events)[i + 1]));
        const int k = (*d->prof_kinds)[i / 2];
        ms[k] += (double)t;
        launches[k] += 1;
    }
    d->prof_used = 0;
    return QMC_OK;
}

extern "C" int qmc_det_info(const qmc_det_t *d, int *nw, int *nel, int *ld, int *delay_rank)
{
    QMC_REQUIRE(d, "qmc_det_info: NULL handle");
    if (nw) *nw = d->nw;
    if (nel) *nel = d->nel;
    if (ld) *ld = d->ld;
    if (delay_rank) *delay_rank = d->delay;
    return QMC_OK;
}

extern "C" int qmc_det_storage(const qmc_det_t *d, int *bytes_per_element)
{
    QMC_REQUIRE(d && bytes_per_element, "qmc_det_storage: NULL argument");
    *bytes_per_element = d->b32 ? 4 : 8;
    return QMC_OK;
}

extern "C" int qmc_det_recompute(qmc_det_t *d, const qmc_spline_t *sp, const double *pos, void *stream)
{
    QMC_REQUIRE(d && sp && pos, "qmc_det_recompute: NULL argument");
    QMC_REQUIRE(d->spline == sp, "qmc_det_recompute: the determinant was initialised from another spline");
    cudaStream_t s = (cudaStream_t)stream;
    int rc = qmc_det_flush(d, stream);               // closes an open window (its rows are superseded anyway)
    if (rc) return rc;
    init_stats_kernel<<<(d->nw + 127) / 128, 128, 0, s>>>(d->nw, d->logdet, d->sign, nullptr);
    QMC_LAUNCHED();
    bool singular = false;
    rc = build_inverse(d, sp, pos, s, &singular);
    if (rc) return rc;
    return singular ? QMC_ESINGULAR : QMC_OK;
}

namespace qmc {

// pos[w][iel_s] of the sampled electrons iel_s = s * stride, packed as [ns][nw][3].
__global__ void gather_sample_pos_kernel(const double *__restrict__ pos, int nw, int nel, int ns, int stride,
                                         double *__restrict__ out)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= ns * nw) return;
    const int sidx = e / nw, w = e % nw;
    const double *r = pos + ((size_t)w * nel + (size_t)sidx * stride) * 3;
    out[3 * (size_t)e + 0] = r[0]; out[3 * (size_t)e + 1] = r[1]; out[3 * (size_t)e + 2] = r[2];
}

// resid[w] = max over the sampled electrons i and all rows k of |B[k] . phi(r_i) - delta_ik|: rows of
// A B^T - I (= columns of the residual of the inverse).  Grid (row chunks of 64, walkers); one warp per
// row, the sampled orbital vectors in shared memory (fp64); the max of non-negative doubles is taken
// with an integer atomicMax on their bit patterns (order-independent, hence reproducible).
template <typename TB>
__global__ void __launch_bounds__(256)
residual_kernel(const TB *__restrict__ B, int nel, int ld, int np, int nw, int ns, int stride,
                const float *__restrict__ phi /* [ns][nw][np] */, double *__restrict__ resid)
{
    extern __shared__ double phi_s[];                 // [ns][nel]
    const int w = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int e = threadIdx.x; e < ns * nel; e += 256) {
        const int sidx = e / nel, j = e % nel;
        phi_s[e] = (double)phi[((size_t)sidx * nw + w) * np + j];
    }
    __syncthreads();
    double worst = 0.0;
    const int k_end = min(nel, (int)(blockIdx.x + 1) * 64);
    for (int k = blockIdx.x * 64 + warp; k < k_end; k += 8) {
        const TB *row = B + ((size_t)w * nel + k) * ld;
        for (int sidx = 0; sidx < ns; ++sidx) {
            double acc = 0.0;
            for (int j = lane; j < nel; j += 32) acc = fma((double)row[j], phi_s[sidx * nel + j], acc);
            acc = warp_sum(acc);
            const double r = fabs(acc - (k == sidx * stride ? 1.0 : 0.0));
            worst = (r > worst || r != r) ? (r != r ? __longlong_as_double(0x7ff0000000000000LL) : r) : worst;   // NaN counts as +inf
        }
    }
    if (lane == 0) atomicMax(reinterpret_cast<unsigned long long *>(resid + w), (unsigned long long)__double_as_longlong(worst));
}

}  // namespace qmc

extern "C" int qmc_det_residual(qmc_det_t *d, const qmc_spline_t *sp, const double *pos, int nsample,
                                double *resid_out, void *stream)
{
    QMC_REQUIRE(d && sp && pos && resid_out, "qmc_det_residual: NULL argument");
    QMC_REQUIRE(d->spline == sp, "qmc_det_residual: the determinant was initialised from another spline");
    QMC_REQUIRE(nsample >= 1 && nsample <= d->nel, "qmc_det_residual: nsample=%d not in 1..%d", nsample, d->nel);
    const int nw = d->nw, nel = d->nel, np = d->np, stride = nel / nsample;
    const size_t smem = (size_t)nsample * nel * sizeof(double);
    QMC_REQUIRE(smem <= 96 * 1024, "qmc_det_residual: nsample=%d needs %zu bytes of shared memory (max 96 KB)", nsample, smem);
    cudaStream_t s = (cudaStream_t)stream;
    int rc = qmc_det_flush(d, stream);
    if (rc) return rc;
    double *spos = nullptr;
    float *phi = nullptr;
    if ((rc = dev_alloc(&spos, (size_t)nsample * nw * 3, "sample positions"))) return rc;
    if ((rc = dev_alloc(&phi, (size_t)nsample * nw * np, "sample orbitals"))) { cudaFree(spos); return rc; }
    gather_sample_pos_kernel<<<(nsample * nw + 127) / 128, 128, 0, s>>>(pos, nw, nel, nsample, stride, spos);
    count_launch();
    rc = qmc_spo_vgl(sp, nsample * nw, spos, phi, nullptr, nullptr, np, s);
    cudaError_t e = cudaSuccess;
    if (!rc) {
        e = cudaMemsetAsync(resid_out, 0, (size_t)nw * sizeof(double), s);
        dim3 grid((nel + 63) / 64, nw);
        if (e == cudaSuccess) {
            QMC_WITH_B(d, TB, Bp, {
                e = cudaFuncSetAttribute(residual_kernel<TB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
                if (e == cudaSuccess)
                    residual_kernel<TB><<<grid, 256, smem, s>>>(Bp, nel, d->ld, np, nw, nsample, stride, phi, resid_out);
            });
            count_launch();
        }
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);       // the scratch is freed below
    }
    cudaFree(spos);
    cudaFree(phi);
    if (rc) return rc;
    if (e != cudaSuccess) { set_error("qmc_det_residual: %s", cudaGetErrorString(e)); return QMC_ECUDA; }
    return QMC_OK;
}

extern "C" int qmc_det_ratio(qmc_det_t *d, int iel, const float *phi, int ldo, double *ratio, void *stream)
{
    QMC_REQUIRE(d && phi && ratio, "qmc_det_ratio: NULL argument");
    QMC_REQUIRE(iel >= 0 && iel < d->nel, "qmc_det_ratio: iel=%d out of range 0..%d", iel, d->nel - 1);
    QMC_REQUIRE(ldo >= d->nel, "qmc_det_ratio: ldo=%d < nel=%d", ldo, d->nel);
    cudaStream_t s = (cudaStream_t)stream;
    if (d->delay) return delayed_ratio(d, iel, phi, ldo, ratio, s);
    QMC_WITH_B(d, TB, Bp, (ratio_kernel<TB><<<d->nw, 128, 0, s>>>(Bp, d->nel, d->ld, iel, phi, ldo, ratio)));
    QMC_LAUNCHED();
    return QMC_OK;
}

extern "C" int qmc_det_ratio_points(qmc_det_t *d, int iel, int npts, const float *phi, int ldo, double *ratios,
                                    void *stream)
{
    QMC_REQUIRE(d && phi && ratios, "qmc_det_ratio_points: NULL argument");
    QMC_REQUIRE(iel >= 0 && iel < d->nel, "qmc_det_ratio_points: iel=%d out of range 0..%d", iel, d->nel - 1);
    QMC_REQUIRE(npts >= 0, "qmc_det_ratio_points: npts=%d", npts);
    QMC_REQUIRE(ldo >= d->nel, "qmc_det_ratio_points: ldo=%d < nel=%d", ldo, d->nel);
    if (npts == 0) return QMC_OK;
    cudaStream_t s = (cudaStream_t)stream;
    if (d->delay) {               // ratios against the current inverse: apply pending rows first
        int rc = delayed_flush_reset_host(d, s);
        if (rc) return rc;
    }
    QMC_WITH_B(d, TB, Bp, (ratio_points_kernel<TB><<<d->nw, 256, 0, s>>>(Bp, d->nel, d->ld, iel, phi, npts, ldo, ratios)));
    QMC_LAUNCHED();
    return QMC_OK;
}

extern "C" int qmc_det_accept_update(qmc_det_t *d, int iel, const float *phi, int ldo, const double *ratio,
                                     const unsigned char *accept, void *stream)
{
    QMC_REQUIRE(d && phi && ratio && accept, "qmc_det_accept_update: NULL argument");
    QMC_REQUIRE(iel >= 0 && iel < d->nel, "qmc_det_accept_update: iel=%d out of range 0..%d", iel, d->nel - 1);
    QMC_REQUIRE(ldo >= d->nel, "qmc_det_accept_update: ldo=%d < nel=%d", ldo, d->nel);
    cudaStream_t s = (cudaStream_t)stream;
    if (d->delay) return delayed_accept(d, iel, phi, ldo, ratio, accept, s);
    QMC_WITH_B(d, TB, Bp, (copy_rowk_kernel<TB><<<d->nw, 256, 0, s>>>(Bp, d->nel, d->ld, iel, accept, d->rowk)));
    QMC_LAUNCHED();
    UpdateArgs a{};
    a.B = d->b32 ? (void *)d->Bf : (void *)d->B; a.nel = d->nel; a.ld = d->ld; a.iel = iel;
    a.phi = phi; a.ldphi = (size_t)ldo; a.rowk = d->rowk;
    a.ratio = ratio; a.accept = accept;
    a.logdet = d->logdet; a.sign = d->sign; a.naccept = d->naccept;
    const cudaError_t ue = d->b32 ? launch_sm_update<float, false>(a, d->nw, s) : launch_sm_update<double, false>(a, d->nw, s);
    QMC_CUDA(ue);
    return QMC_OK;
}

extern "C" int qmc_det_flush(qmc_det_t *d, void *stream)
{
    QMC_REQUIRE(d, "qmc_det_flush: NULL handle");
    if (!d->delay) return QMC_OK;
    return delayed_flush_reset_host(d, (cudaStream_t)stream);
}

extern "C" int qmc_det_get_inverse(qmc_det_t *d, double *out, void *stream)
{
    QMC_REQUIRE(d && out, "qmc_det_get_inverse: NULL argument");
    int rc = qmc_det_flush(d, stream);
    if (rc) return rc;
    QMC_WITH_B(d, TB, Bp, (pack_inverse_kernel<TB, true><<<d->nw * d->nel, 256, 0, (cudaStream_t)stream>>>(Bp, out, d->nel, d->ld)));
    QMC_LAUNCHED();
    return QMC_OK;
}

extern "C" int qmc_det_set_inverse(qmc_det_t *d, const double *in, const double *logdet, const int *sign,
                                   void *stream)
{
    QMC_REQUIRE(d && in, "qmc_det_set_inverse: NULL argument");
    cudaStream_t s = (cudaStream_t)stream;
    int rc = qmc_det_flush(d, stream);
    if (rc) return rc;
    QMC_WITH_B(d, TB, Bp, (pack_inverse_kernel<TB, false><<<d->nw * d->nel, 256, 0, s>>>(Bp, const_cast<double *>(in), d->nel, d->ld)));
    QMC_LAUNCHED();
    if (logdet) QMC_CUDA(cudaMemcpyAsync(d->logdet, logdet, (size_t)d->nw * sizeof(double), cudaMemcpyDeviceToDevice, s));
    if (sign) QMC_CUDA(cudaMemcpyAsync(d->sign, sign, (size_t)d->nw * sizeof(int), cudaMemcpyDeviceToDevice, s));
    return QMC_OK;
}

extern "C" int qmc_det_get_stats(qmc_det_t *d, double *logdet, int *sign, long long *naccept, void *stream)
{
    QMC_REQUIRE(d, "qmc_det_get_stats: NULL handle");
    cudaStream_t s = (cudaStream_t)stream;
    if (logdet) QMC_CUDA(cudaMemcpyAsync(logdet, d->logdet, (size_t)d->nw * sizeof(double), cudaMemcpyDeviceToDevice, s));
    if (sign) QMC_CUDA(cudaMemcpyAsync(sign, d->sign, (size_t)d->nw * sizeof(int), cudaMemcpyDeviceToDevice, s));
    if (naccept) QMC_CUDA(cudaMemcpyAsync(naccept, d->naccept, (size_t)d->nw * sizeof(long long), cudaMemcpyDeviceToDevice, s));
    return QMC_OK;
}
