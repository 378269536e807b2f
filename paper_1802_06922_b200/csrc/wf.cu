// qmc_wf_*: the product of two spin determinants, Psi_T = D_up D_dn (eq. 26, with one
// determinant per spin, c_1 = 1; a Jastrow factor is an option of the sweep, qmc_sweep_opts_t.jastrow).  A particle-by-particle sweep iterates
// "sequentially over all electrons" (L195): the N_up electrons of the up determinant, then the N_dn of
// the down determinant.  Moving an up electron leaves D_dn unchanged, so the ratio of the move is
// D_up'/D_up and only the up inverse is updated (and vice versa): the sweep is the up sweep followed
// by the down sweep, each on its own handle, orbitals and half of the move arrays.  The kinetic term of
// the local energy is the sum of the two determinants' terms (eq. 3: a sum over electrons).
#include <new>

#include "common.cuh"

struct qmc_wf {
    qmc_det *det[2];
    const qmc_spline *spline[2];
    double *scratch;          // [2][nw] for qmc_wf_kinetic / qmc_wf_get_stats
    int *iscratch;            // [2][nw]
};

namespace qmc {

__global__ void wf_add_kernel(int nw, const double *a, const double *b, double *out)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < nw) out[w] = a[w] + b[w];
}
__global__ void wf_sign_kernel(int nw, const int *a, const int *b, int *out)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < nw) out[w] = a[w] * b[w];
}

}  // namespace qmc

using namespace qmc;

extern "C" int qmc_wf_create(qmc_wf_t **out, qmc_det_t *det_up, const qmc_spline_t *spline_up, qmc_det_t *det_dn,
                             const qmc_spline_t *spline_dn)
{
    QMC_REQUIRE(out && det_up && spline_up && det_dn && spline_dn, "qmc_wf_create: NULL argument");
    *out = nullptr;
    QMC_REQUIRE(det_up != det_dn, "qmc_wf_create: the two determinants must be different handles");
    QMC_REQUIRE(det_up->spline == spline_up && det_dn->spline == spline_dn,
                "qmc_wf_create: a determinant was initialised from another spline");
    QMC_REQUIRE(det_up->nw == det_dn->nw, "qmc_wf_create: walker counts differ (%d, %d)", det_up->nw, det_dn->nw);
    QMC_REQUIRE(det_up->device == det_dn->device, "qmc_wf_create: the determinants live on different devices");
    qmc_wf *wf = new (std::nothrow) qmc_wf();
    if (!wf) { set_error("qmc_wf_create: host allocation failed"); return QMC_ENOMEM; }
    wf->det[0] = det_up; wf->det[1] = det_dn;
    wf->spline[0] = spline_up; wf->spline[1] = spline_dn;
    const size_t nw = (size_t)det_up->nw;
    if (cudaMalloc((void **)&wf->scratch, 2 * nw * sizeof(double)) != cudaSuccess ||
        cudaMalloc((void **)&wf->iscratch, 2 * nw * sizeof(int)) != cudaSuccess) {
        (void)cudaGetLastError();
        cudaFree(wf->scratch);
        delete wf;
        set_error("qmc_wf_create: device allocation failed");
        return QMC_ENOMEM;
    }
    *out = wf;
    return QMC_OK;
}

extern "C" int qmc_wf_destroy(qmc_wf_t *wf)
{
    if (!wf) return QMC_OK;
    cudaFree(wf->scratch);
    cudaFree(wf->iscratch);
    delete wf;
    return QMC_OK;
}

extern "C" int qmc_wf_info(const qmc_wf_t *wf, int *nwalkers, int *nup, int *ndn)
{
    QMC_REQUIRE(wf, "qmc_wf_info: NULL handle");
    if (nwalkers) *nwalkers = wf->det[0]->nw;
    if (nup) *nup = wf->det[0]->nel;
    if (ndn) *ndn = wf->det[1]->nel;
    return QMC_OK;
}

extern "C" int qmc_wf_sweep(qmc_wf_t *wf, double *pos_up, double *pos_dn, const double *delta, const double *unif,
                            int nsweeps, double *ratios_out, unsigned char *accept_out, const unsigned char *forced,
                            const qmc_sweep_opts_t *opts, void *stream)
{
    QMC_REQUIRE(wf && pos_up && pos_dn && delta && unif, "qmc_wf_sweep: NULL argument");
    QMC_REQUIRE(nsweeps >= 0, "qmc_wf_sweep: nsweeps=%d", nsweeps);
    QMC_REQUIRE(!opts || (opts->iel_begin == 0 && opts->iel_count == 0 && !opts->phi_record),
                "qmc_wf_sweep: iel_begin / iel_count / phi_record are per-determinant options (use qmc_sweep_ex)");
    const size_t nw = (size_t)wf->det[0]->nw, nup = (size_t)wf->det[0]->nel, ndn = (size_t)wf->det[1]->nel, n = nup + ndn;
    double *pos[2] = {pos_up, pos_dn};
    for (int sw = 0; sw < nsweeps; ++sw) {
        for (int sp = 0; sp < 2; ++sp) {
            const size_t mv = ((size_t)sw * n + (sp ? nup : 0)) * nw;      // first move of this spin in this sweep
            qmc_sweep_opts_t o{};
            if (opts) {
                o = *opts;
                if (o.force_out) o.force_out += 3 * mv;
                if (o.rprop_out) o.rprop_out += 3 * mv;
                if (o.fcur_out) o.fcur_out += 3 * mv;
                if (o.logt_out) o.logt_out += mv;
                if (o.jastrow) {          // the other spin's electrons, where they are now, are the fixed particles
                    o.jastrow_other = pos[1 - sp];
                    o.jastrow_nother = wf->det[1 - sp]->nel;
                    if (o.jratio_out) o.jratio_out += mv;
                }
            }
            int rc = qmc_sweep_ex(wf->det[sp], wf->spline[sp], pos[sp], delta + 3 * mv, unif + mv, 1,
                                  ratios_out ? ratios_out + mv : nullptr, accept_out ? accept_out + mv : nullptr,
                                  forced ? forced + mv : nullptr, opts ? &o : nullptr, stream);
            if (rc) return rc;
        }
    }
    return QMC_OK;
}

extern "C" int qmc_wf_kinetic(qmc_wf_t *wf, const double *pos_up, const double *pos_dn, double *ekin_out, void *stream)
{
    QMC_REQUIRE(wf && pos_up && pos_dn && ekin_out, "qmc_wf_kinetic: NULL argument");
    const int nw = wf->det[0]->nw;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = qmc_det_kinetic(wf->det[0], wf->spline[0], pos_up, nullptr, nullptr, nullptr, wf->scratch, stream);
    if (rc) return rc;
    rc = qmc_det_kinetic(wf->det[1], wf->spline[1], pos_dn, nullptr, nullptr, nullptr, wf->scratch + nw, stream);
    if (rc) return rc;
    wf_add_kernel<<<(nw + 127) / 128, 128, 0, s>>>(nw, wf->scratch, wf->scratch + nw, ekin_out);
    QMC_LAUNCHED();
    return QMC_OK;
}

extern "C" int qmc_wf_get_stats(qmc_wf_t *wf, double *logpsi, int *sign, void *stream)
{
    QMC_REQUIRE(wf, "qmc_wf_get_stats: NULL handle");
    const int nw = wf->det[0]->nw;
    cudaStream_t s = (cudaStream_t)stream;
    for (int sp = 0; sp < 2; ++sp) {
        int rc = qmc_det_get_stats(wf->det[sp], wf->scratch + (size_t)sp * nw, wf->iscratch + (size_t)sp * nw, nullptr, stream);
        if (rc) return rc;
    }
    if (logpsi) { wf_add_kernel<<<(nw + 127) / 128, 128, 0, s>>>(nw, wf->scratch, wf->scratch + nw, logpsi); QMC_LAUNCHED(); }
    if (sign) { wf_sign_kernel<<<(nw + 127) / 128, 128, 0, s>>>(nw, wf->iscratch, wf->iscratch + nw, sign); QMC_LAUNCHED(); }
    return QMC_OK;
}
