// qmc_jastrow_*: one- and two-body B-spline Jastrow factor (sec 7: eq. 28-29 Psi = e^{-J} Phi,
// eq. 30 many-body expansion, eq. 31 one-body term, eq. 32 first term, eq. 33 the cubic B-spline
// functor), as far as the particle-by-particle move needs it: the ratio exp(-dJ) of a single-electron
// move, batched over walkers and over the steps of a delayed window, and J itself for checks.
#include <math.h>

#include <new>

#include "jastrow_device.cuh"

namespace qmc {

struct JasMoveArgs {
    const JasTable *table;
    int nion;
    const double *ion;        // [nion][3]
    const int *ion_func;      // [nion]
    int nw, nel, nother;
    const double *pos;        // [nw][nel][3] the swept electrons (one spin)
    const double *other;      // [nw][nother][3] electrons of the other spin, or NULL
    int iel0;                 // step j of the batch moves electron iel0 + j
    const double *delta;      // [nb][nw][3] displacements (r' = pos + delta), or NULL
    const double *rnew;       // [nw][3] explicit proposals (one step), used when delta == NULL
    double *dj_out;           // [nb][nw] or NULL
    double *ratio_out;        // [nb][nw] exp(-dJ) or NULL
    double *tfac_out;         // [nb][nw] exp(-2 dJ) or NULL
    double *corr_out;         // [nw][ncorr][ncorr] or NULL: corr[w][j][m], m < j: what the ACCEPTED move of step m
    int ncorr;                //   (earlier in the same batch) adds to dJ of step j -- the same-spin pair term with
                              //   electron iel0 + m at its proposed instead of its old position
    const int *cur;           // accept windows: step j moves electron cur[w] + j (nothing beyond kend) and delta is
    int kend;                 //   offset to (sweep, electron 0) and indexed with the electron
};

constexpr int kJasThreads = 128;

// dJ of the move of electron iel0 + j of walker w with every other particle where `pos` / `other` /
// the ions put it: the terms of eq. 30 that contain the moved electron.  One block per (walker, step);
// thread t sums particles t, t + 128, ... in order, then a fixed-order block sum.
__global__ void __launch_bounds__(kJasThreads) jastrow_move_kernel(JasMoveArgs a)
{
    __shared__ JasTable T;
    __shared__ double red[33];
    const int w = blockIdx.x, j = blockIdx.y;
    const int first = a.cur ? a.cur[w] : a.iel0, k = first + j;
    if (a.cur && k >= a.kend) return;                      // beyond this walker's sweep (block-uniform, before any barrier)
    {
        const int *src = reinterpret_cast<const int *>(a.table);
        int *dst = reinterpret_cast<int *>(&T);
        for (int i = threadIdx.x; i < (int)(sizeof(JasTable) / sizeof(int)); i += kJasThreads) dst[i] = src[i];
    }
    __syncthreads();
    const int jd0 = a.cur ? first : 0;                     // delta index of step 0
    const double *pw = a.pos + (size_t)w * a.nel * 3;
    const double rold[3] = {pw[3 * k], pw[3 * k + 1], pw[3 * k + 2]};
    double rnew[3];
    if (a.delta) {
        const double *dl = a.delta + 3 * ((size_t)(jd0 + j) * a.nw + w);
        rnew[0] = rold[0] + dl[0]; rnew[1] = rold[1] + dl[1]; rnew[2] = rold[2] + dl[2];
    } else {
        rnew[0] = a.rnew[3 * (size_t)w]; rnew[1] = a.rnew[3 * (size_t)w + 1]; rnew[2] = a.rnew[3 * (size_t)w + 2];
    }
    double s = 0.0;
    for (int i = threadIdx.x; i < a.nel; i += kJasThreads)
        if (i != k) s += jas_pair_delta(T, T.f_same, rnew, rold, pw + 3 * i);
    if (a.other) {
        const double *ow = a.other + (size_t)w * a.nother * 3;
        for (int i = threadIdx.x; i < a.nother; i += kJasThreads) s += jas_pair_delta(T, T.f_opp, rnew, rold, ow + 3 * i);
    }
    for (int i = threadIdx.x; i < a.nion; i += kJasThreads) s += jas_pair_delta(T, a.ion_func[i], rnew, rold, a.ion + 3 * i);
    if (a.corr_out && (int)threadIdx.x < j) {
        const int m = threadIdx.x;
        const double *ro_m = pw + 3 * (first + m);
        const double *dm = a.delta + 3 * ((size_t)(jd0 + m) * a.nw + w);
        const double rn_m[3] = {ro_m[0] + dm[0], ro_m[1] + dm[1], ro_m[2] + dm[2]};
        a.corr_out[((size_t)w * a.ncorr + j) * a.ncorr + m] =
            jas_pair_delta(T, T.f_same, rnew, rold, rn_m) - jas_pair_delta(T, T.f_same, rnew, rold, ro_m);
    }
    const double dj = block_sum(s, red);
    if (threadIdx.x == 0) {
        const size_t o = (size_t)j * a.nw + w;
        if (a.dj_out) a.dj_out[o] = dj;
        if (a.ratio_out) a.ratio_out[o] = exp(-dj);
        if (a.tfac_out) a.tfac_out[o] = exp(-2.0 * dj);
    }
}

// J of eq. 30 (one- and two-body terms) of every walker: one block per walker.
__global__ void __launch_bounds__(256) jastrow_value_kernel(const JasTable *table, int nion, const double *ion,
                                                            const int *ion_func, int nel, const double *pos, int nother,
                                                            const double *other, double *out)
{
    __shared__ JasTable T;
    __shared__ double red[33];
    {
        const int *src = reinterpret_cast<const int *>(table);
        int *dst = reinterpret_cast<int *>(&T);
        for (int i = threadIdx.x; i < (int)(sizeof(JasTable) / sizeof(int)); i += 256) dst[i] = src[i];
    }
    __syncthreads();
    const int w = blockIdx.x, n = nel + nother;
    const double *pw = pos + (size_t)w * nel * 3;
    const double *ow = other ? other + (size_t)w * nother * 3 : nullptr;
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += 256) {
        const double *ri = i < nel ? pw + 3 * i : ow + 3 * (i - nel);
        for (int I = 0; I < nion; ++I) s += jas_u(T, ion_func[I], jas_dist(T, ri, ion + 3 * I));
        for (int j = i + 1; j < n; ++j) {             // each unordered pair once = 1/2 sum over i != j
            const double *rj = j < nel ? pw + 3 * j : ow + 3 * (j - nel);
            s += jas_u(T, (i < nel) == (j < nel) ? T.f_same : T.f_opp, jas_dist(T, ri, rj));
        }
    }
    s = block_sum(s, red);
    if (threadIdx.x == 0) out[w] = s;
}

// Enqueue dJ / exp(-dJ) / exp(-2 dJ) of a batch of nb consecutive steps (sweep.cu, window path) or of one
// step with explicit proposals.
int jastrow_move_launch(const qmc_jastrow *J, int nw, int nel, const double *pos, int nother, const double *other,
                        int iel0, int nb, const double *delta, const double *rnew, double *dj_out, double *ratio_out,
                        double *tfac_out, double *corr_out, int ncorr, cudaStream_t s, const int *cur, int kend)
{
    JasMoveArgs a{};
    a.table = J->table; a.nion = J->nion; a.ion = J->ion; a.ion_func = J->ion_func;
    a.nw = nw; a.nel = nel; a.nother = other ? nother : 0;
    a.pos = pos; a.other = other; a.iel0 = iel0; a.delta = delta; a.rnew = rnew;
    a.dj_out = dj_out; a.ratio_out = ratio_out; a.tfac_out = tfac_out;
    a.corr_out = delta ? corr_out : nullptr; a.ncorr = ncorr;
    a.cur = cur; a.kend = kend;
    jastrow_move_kernel<<<dim3(nw, nb), kJasThreads, 0, s>>>(a);
    QMC_LAUNCHED();
    return QMC_OK;
}

}  // namespace qmc

using namespace qmc;

static bool invert3(const double L[9], double Li[9])
{
    const double det = L[0] * (L[4] * L[8] - L[5] * L[7]) - L[1] * (L[3] * L[8] - L[5] * L[6]) + L[2] * (L[3] * L[7] - L[4] * L[6]);
    if (det == 0.0 || !isfinite(det)) return false;
    const double id = 1.0 / det;
    Li[0] = (L[4] * L[8] - L[5] * L[7]) * id; Li[1] = (L[2] * L[7] - L[1] * L[8]) * id; Li[2] = (L[1] * L[5] - L[2] * L[4]) * id;
    Li[3] = (L[5] * L[6] - L[3] * L[8]) * id; Li[4] = (L[0] * L[8] - L[2] * L[6]) * id; Li[5] = (L[2] * L[3] - L[0] * L[5]) * id;
    Li[6] = (L[3] * L[7] - L[4] * L[6]) * id; Li[7] = (L[1] * L[6] - L[0] * L[7]) * id; Li[8] = (L[0] * L[4] - L[1] * L[3]) * id;
    return true;
}

extern "C" int qmc_jastrow_create(qmc_jastrow_t **out, const double *lattice, int nfunc, const double *rc, const int *M,
                                  const double *p, int f_same, int f_opp, int nion, const double *ion_pos,
                                  const int *ion_func)
{
    QMC_REQUIRE(out, "qmc_jastrow_create: NULL argument");
    *out = nullptr;
    QMC_REQUIRE(nfunc >= 1 && nfunc <= kJasMaxFunc && rc && M && p, "qmc_jastrow_create: nfunc=%d (1..%d) or NULL tables", nfunc, kJasMaxFunc);
    QMC_REQUIRE(f_same >= -1 && f_same < nfunc && f_opp >= -1 && f_opp < nfunc, "qmc_jastrow_create: f_same=%d f_opp=%d", f_same, f_opp);
    QMC_REQUIRE(nion >= 0 && (nion == 0 || (ion_pos && ion_func)), "qmc_jastrow_create: nion=%d", nion);
    qmc_jastrow *J = new (std::nothrow) qmc_jastrow();
    if (!J) { set_error("qmc_jastrow_create: host allocation failed"); return QMC_ENOMEM; }
    JasTable &T = J->host;
    T = JasTable{};
    T.nfunc = nfunc; T.f_same = f_same; T.f_opp = f_opp;
    int off = 0, src = 0;
    for (int f = 0; f < nfunc; ++f) {
        if (!(M[f] >= 1 && rc[f] > 0.0 && isfinite(rc[f])) || off + M[f] + 4 > kJasMaxCoef) {
            set_error("qmc_jastrow_create: function %d: M=%d r_c=%g (or more than %d control points in all)", f, M[f], rc[f], kJasMaxCoef);
            delete J;
            return QMC_EINVAL;
        }
        T.rc[f] = rc[f];
        T.dinv[f] = (double)M[f] / rc[f];
        T.off[f] = off;
        for (int m = 0; m <= M[f]; ++m) T.p[off + m] = p[src + m];
        off += M[f] + 4;          // three zeros behind p_M: the sum of eq. 33 stops at M
        src += M[f] + 1;
    }
    if (lattice) {
        for (int i = 0; i < 9; ++i) T.lat[i] = lattice[i];
        if (!invert3(T.lat, T.linv)) { set_error("qmc_jastrow_create: singular lattice"); delete J; return QMC_EINVAL; }
        T.periodic = 1;
        T.ortho = lattice[1] == 0.0 && lattice[2] == 0.0 && lattice[3] == 0.0 && lattice[5] == 0.0 && lattice[6] == 0.0 && lattice[7] == 0.0;
    }
    for (int i = 0; i < nion; ++i)
        if (ion_func[i] < -1 || ion_func[i] >= nfunc) { set_error("qmc_jastrow_create: ion %d has function %d", i, ion_func[i]); delete J; return QMC_EINVAL; }
    J->nion = nion;
    cudaGetDevice(&J->device);
    cudaError_t e = cudaMalloc((void **)&J->table, sizeof(JasTable));
    if (e == cudaSuccess && nion) e = cudaMalloc((void **)&J->ion, (size_t)nion * 3 * sizeof(double));
    if (e == cudaSuccess && nion) e = cudaMalloc((void **)&J->ion_func, (size_t)nion * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(J->table, &T, sizeof(JasTable), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && nion) e = cudaMemcpy(J->ion, ion_pos, (size_t)nion * 3 * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && nion) e = cudaMemcpy(J->ion_func, ion_func, (size_t)nion * sizeof(int), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        set_error("qmc_jastrow_create: %s", cudaGetErrorString(e));
        (void)cudaGetLastError();
        cudaFree(J->table); cudaFree(J->ion); cudaFree(J->ion_func);
        delete J;
        return e == cudaErrorMemoryAllocation ? QMC_ENOMEM : QMC_ECUDA;
    }
    *out = J;
    return QMC_OK;
}

extern "C" int qmc_jastrow_destroy(qmc_jastrow_t *J)
{
    if (!J) return QMC_OK;
    cudaFree(J->table);
    cudaFree(J->ion);
    cudaFree(J->ion_func);
    delete J;
    return QMC_OK;
}

extern "C" int qmc_jastrow_ratio(const qmc_jastrow_t *J, int nwalkers, int nel, const double *pos, int nother,
                                 const double *other, int iel, const double *rnew, double *ratio_out, double *dj_out,
                                 void *stream)
{
    QMC_REQUIRE(J && pos && rnew && (ratio_out || dj_out), "qmc_jastrow_ratio: NULL argument");
    QMC_REQUIRE(nwalkers >= 0 && nel >= 1 && iel >= 0 && iel < nel, "qmc_jastrow_ratio: nwalkers=%d nel=%d iel=%d", nwalkers, nel, iel);
    QMC_REQUIRE(nother >= 0 && (nother == 0 || other), "qmc_jastrow_ratio: nother=%d without positions", nother);
    if (nwalkers == 0) return QMC_OK;
    return jastrow_move_launch(J, nwalkers, nel, pos, nother, nother ? other : nullptr, iel, 1, nullptr, rnew, dj_out,
                               ratio_out, nullptr, nullptr, 0, (cudaStream_t)stream, nullptr, 0);
}

extern "C" int qmc_jastrow_value(const qmc_jastrow_t *J, int nwalkers, int nel, const double *pos, int nother,
                                 const double *other, double *j_out, void *stream)
{
    QMC_REQUIRE(J && pos && j_out, "qmc_jastrow_value: NULL argument");
    QMC_REQUIRE(nwalkers >= 0 && nel >= 1 && nother >= 0 && (nother == 0 || other), "qmc_jastrow_value: nwalkers=%d nel=%d nother=%d", nwalkers, nel, nother);
    if (nwalkers == 0) return QMC_OK;
    jastrow_value_kernel<<<nwalkers, 256, 0, (cudaStream_t)stream>>>(J->table, J->nion, J->ion, J->ion_func, nel, pos, nother,
                                                                     nother ? other : nullptr, j_out);
    QMC_LAUNCHED();
    return QMC_OK;
}
