// qmc_sweep*: the particle-by-particle sweep driver (sec 5.2.1) -- all walkers
// in lockstep (L114, L181), electrons in sequence.  Launches:
//   K1 spo_batch_kernel      S0 proposal, S1 stencil, S2 SPO-VGL gather -- once per batch of steps
//   K2 ratio_rowcopy_kernel  S3 ratio, copy of row k                    -- per electron step
//   K3 sm_update_kernel      S4 Metropolis test, S5 rank-1 update       -- per electron step
// (delayed mode, per window of K steps: K1, then delayed_window_kernel = S3 + S4 of the K steps,
//  then flush_dmma_kernel = S5')
#include "delayed_device.cuh"
#include "spo_device.cuh"
#include "update_device.cuh"

namespace qmc {

void spo_launch_shape(int np, int *threads, int *tiles);

// SPO-VGL of a BATCH of electron steps in one launch.  The proposal of electron k does not depend
// on the outcome of the moves before it (r' = pos[w][k] + delta, and pos[w][k] only changes at step
// k itself), so the gathers of `nb` consecutive steps are issued together: nb * nw positions keep
// every SM streaming (a single step's 512 positions is a 25 us launch that never leaves the ramp).
struct SpoBatchArgs {
    SplineView sp;
    const double *pos;     // [nw][nel][3]
    const double *delta;   // [nb][nw][3], offset to (sweep, first electron of the batch); NULL = the current positions
    int nel, iel0, nw;
    float *vgl;            // [nb][nw][5][np]
    float *phi_record;     // [nb][nrecord][nel], offset to (sweep, first electron), or NULL
    int nrecord;
};

// One block per (orbital tile, walker, step of the batch).  Thread t owns orbitals 4t..4t+3 of the
// tile: it gathers their value/gradient/Laplacian from the 64 stencil rows (S0-S2).
__global__ void __launch_bounds__(256) spo_batch_kernel(SpoBatchArgs a)
{
    __shared__ StencilSmem st;
    const int w = blockIdx.y, j = blockIdx.z;
    const double *r = a.pos + ((size_t)w * a.nel + a.iel0 + j) * 3;
    double dx = 0.0, dy = 0.0, dz = 0.0;
    if (a.delta) {
        const double *dl = a.delta + 3 * ((size_t)j * a.nw + w);
        dx = dl[0]; dy = dl[1]; dz = dl[2];
    }
    stage_stencil(a.sp, r[0] + dx, r[1] + dy, r[2] + dz, st);
    const int np = a.sp.np;
    const int col = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
    if (col >= np) return;
    float4 v, gx, gy, gz, lp;
    gather4<true>(a.sp, st, col, v, gx, gy, gz, lp);
    float *o = a.vgl + ((size_t)j * a.nw + w) * 5 * np + col;
    *reinterpret_cast<float4 *>(o) = v;
    *reinterpret_cast<float4 *>(o + np) = gx;
    *reinterpret_cast<float4 *>(o + 2 * (size_t)np) = gy;
    *reinterpret_cast<float4 *>(o + 3 * (size_t)np) = gz;
    *reinterpret_cast<float4 *>(o + 4 * (size_t)np) = lp;
    if (a.phi_record && w < a.nrecord) {
        float *rec = a.phi_record + ((size_t)j * a.nrecord + w) * a.nel;
        if (col + 0 < a.nel) rec[col + 0] = v.x;
        if (col + 1 < a.nel) rec[col + 1] = v.y;
        if (col + 2 < a.nel) rec[col + 2] = v.z;
        if (col + 3 < a.nel) rec[col + 3] = v.w;
    }
}

// S3 for the rank-1 path: R_w = B_w[iel] . phi_w (fp64, fixed order) and a copy of row iel, so that
// the update kernel can overwrite B in place.  One block per walker.  With force_out the three
// gradient vectors of the proposal (phi + np, + 2 np, + 3 np) are contracted with the same row:
// F = 2 grad log Psi_T at the proposed configuration = 2 (B[iel] . grad phi) / R.
template <typename TB>
__global__ void __launch_bounds__(256)
ratio_rowcopy_kernel(const TB *__restrict__ B, int nel, int ld, int iel, const float *__restrict__ phi,
                     size_t ldphi, int np, double *__restrict__ rowk, double *__restrict__ ratio,
                     double *__restrict__ force_out)
{
    __shared__ double red[33];
    const int w = blockIdx.x;
    const TB *row = B + ((size_t)w * nel + iel) * ld;
    const float *pw = phi + (size_t)w * ldphi;
    const float2 *ph = reinterpret_cast<const float2 *>(pw);
    double2 *dst = reinterpret_cast<double2 *>(rowk + (size_t)w * ld);
    double acc = 0.0, g[3] = {0.0, 0.0, 0.0};
    for (int j = threadIdx.x; j < ld / 2; j += 256) {
        const double2 b = ld2(row + 2 * j);
        dst[j] = b;
        if (2 * j < nel) {          // phi is padded with zeros up to the table pitch >= nel
            const float2 f = ph[j];
            acc = fma(b.x, (double)f.x, acc);
            acc = fma(b.y, (double)f.y, acc);
            if (force_out) {
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const float2 q = reinterpret_cast<const float2 *>(pw + (size_t)(1 + d) * np)[j];
                    g[d] = fma(b.x, (double)q.x, g[d]);
                    g[d] = fma(b.y, (double)q.y, g[d]);
                }
            }
        }
    }
    acc = block_sum(acc, red);
    if (threadIdx.x == 0) ratio[w] = acc;
    if (force_out) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double gd = block_sum(g[d], red);
            if (threadIdx.x == 0) force_out[3 * (size_t)w + d] = acc != 0.0 ? 2.0 * gd / acc : 0.0;
        }
    }
}

int spo_batch_vgl(qmc_det *d, const qmc_spline *sp, const double *pos, const double *delta, int iel0, int nb,
                  float *phi_record, int nrecord, float *out, cudaStream_t s)
{
    int threads, tiles;
    spo_launch_shape(d->np, &threads, &tiles);
    SpoBatchArgs a{};
    a.sp = sp->view;
    a.pos = pos; a.delta = delta;
    a.nel = d->nel; a.iel0 = iel0; a.nw = d->nw;
    a.vgl = out;
    a.phi_record = phi_record; a.nrecord = nrecord;
    prof_start(d, kProfSpoRatio, s);
    spo_batch_kernel<<<dim3(tiles, d->nw, nb), threads, 0, s>>>(a);
    prof_stop(d, s);
    QMC_LAUNCHED();
    return QMC_OK;
}

// Delayed mode: per window of K consecutive electron steps, K1 (SPO-VGL of the window's proposals),
// delayed_window_kernel (S3 + S4 of the K steps) and the flush (S5').  The proposals of window i+1
// are r' = pos[w][k] + delta for electrons no earlier window of this sweep touches, so K1 of window
// i+1 is enqueued on a second stream as soon as the window kernel of window i has been enqueued and
// runs UNDER the flush of window i (the flush is bound by the fp64 tensor pipe at ranks >= 24 and
// leaves HBM bandwidth unused; the gather is a pure HBM stream).  Two SPO-VGL buffers alternate: buffer
// b is rewritten only after the flush that read it (two windows earlier on `s`) has been enqueued before
// the event the second stream waits on.  Everything the second stream did is joined back into `s`
// before this function returns (the last SPO-VGL is awaited by the last window kernel).
static int sweep_delayed(qmc_det *d, const qmc_spline *sp, double *pos, const double *delta, const double *unif,
                         int nsweeps, int k0, int kn, double *ratios_out, unsigned char *accept_out,
                         const unsigned char *forced, int fixed_node, double *force, float *rec, int nrec,
                         cudaStream_t s)
{
    const int nw = d->nw, nel = d->nel, batch = d->spo_batch;
    const int wins_per_sweep = (kn + batch - 1) / batch;
    const long long nwin = (long long)nsweeps * wins_per_sweep;
    if (nwin == 0) return QMC_OK;
    bool overlap = d->overlap && !d->prof_on;     // per-kernel event timing needs the kernels one after another
    if (overlap && !d->aux) {
        QMC_CUDA(cudaStreamCreateWithFlags(&d->aux, cudaStreamNonBlocking));
        QMC_CUDA(cudaEventCreateWithFlags(&d->ev_spo[0], cudaEventDisableTiming));
        QMC_CUDA(cudaEventCreateWithFlags(&d->ev_spo[1], cudaEventDisableTiming));
        QMC_CUDA(cudaEventCreateWithFlags(&d->ev_main, cudaEventDisableTiming));
    }
    auto spo = [&](long long i, cudaStream_t st) -> int {     // K1 of window i into buffer i & 1
        const int sw = (int)(i / wins_per_sweep), k = k0 + (int)(i % wins_per_sweep) * batch;
        const int nb = min(batch, k0 + kn - k);
        const size_t mv = ((size_t)sw * nel + k) * nw;
        return spo_batch_vgl(d, sp, pos, delta + 3 * mv, k, nb, rec ? rec + mv / nw * (size_t)nrec * nel : nullptr,
                             nrec, d->vgl_buf[overlap ? (i & 1) : 0], st);
    };
    int rc;
    if (overlap) {
        QMC_CUDA(cudaEventRecord(d->ev_main, s));
        QMC_CUDA(cudaStreamWaitEvent(d->aux, d->ev_main, 0));
        if ((rc = spo(0, d->aux))) return rc;
        QMC_CUDA(cudaEventRecord(d->ev_spo[0], d->aux));
    }
    for (long long i = 0; i < nwin; ++i) {
        const int sw = (int)(i / wins_per_sweep), k = k0 + (int)(i % wins_per_sweep) * batch;
        const int nb = min(batch, k0 + kn - k);
        const size_t mv = ((size_t)sw * nel + k) * nw;
        if (overlap) QMC_CUDA(cudaStreamWaitEvent(s, d->ev_spo[i & 1], 0));
        else if ((rc = spo(i, s))) return rc;
        d->vgl = d->vgl_buf[overlap ? (i & 1) : 0];
        rc = delayed_sweep_window(d, pos, delta + 3 * mv, unif + mv, k, nb, ratios_out ? ratios_out + mv : nullptr,
                                  accept_out ? accept_out + mv : nullptr, forced ? forced + mv : nullptr, fixed_node,
                                  force ? force + 3 * mv : nullptr, overlap && i + 1 < nwin ? 1 : 0, s);
        if (rc) return rc;
        if (overlap && i + 1 < nwin) {
            // (delayed_sweep_window recorded ev_main between its window kernel and its flush)
            QMC_CUDA(cudaStreamWaitEvent(d->aux, d->ev_main, 0));
            if ((rc = spo(i + 1, d->aux))) return rc;
            QMC_CUDA(cudaEventRecord(d->ev_spo[(i + 1) & 1], d->aux));
        }
    }
    d->vgl = d->vgl_buf[0];
    return QMC_OK;
}

static int sweep_impl(qmc_det *d, const qmc_spline *sp, double *pos, const double *delta, const double *unif,
                      int nsweeps, double *ratios_out, unsigned char *accept_out, const unsigned char *forced,
                      const qmc_sweep_opts_t *opts, cudaStream_t s)
{
    QMC_REQUIRE(d && sp && pos && delta && unif, "qmc_sweep: NULL argument");
    QMC_REQUIRE(d->spline == sp, "qmc_sweep: the determinant was initialised from another spline");
    QMC_REQUIRE(nsweeps >= 0, "qmc_sweep: nsweeps=%d", nsweeps);
    const int nw = d->nw, nel = d->nel;
    int k0 = 0, kn = nel;
    float *rec = nullptr;
    int nrec = 0, fixed_node = 0;
    double *force = nullptr;
    if (opts) {
        fixed_node = opts->fixed_node != 0;
        force = opts->force_out;
        k0 = opts->iel_begin;
        kn = opts->iel_count ? opts->iel_count : nel - k0;
        rec = opts->phi_record;
        nrec = rec ? opts->nrecord : 0;
        QMC_REQUIRE(k0 >= 0 && kn >= 0 && k0 + kn <= nel, "qmc_sweep_ex: electron range %d+%d outside 0..%d", k0, kn, nel);
        QMC_REQUIRE(nrec >= 0 && nrec <= nw, "qmc_sweep_ex: nrecord=%d outside 0..%d", nrec, nw);
    }
    const int batch = d->spo_batch;
    const size_t slot_stride = (size_t)nw * 5 * d->np;
    if (d->delay) return sweep_delayed(d, sp, pos, delta, unif, nsweeps, k0, kn, ratios_out, accept_out, forced,
                                       fixed_node, force, rec, nrec, s);
    for (int sw = 0; sw < nsweeps; ++sw) {
        for (int k = k0; k < k0 + kn; ++k) {
            const size_t mv = ((size_t)sw * nel + k) * nw;
            const int slot = (k - k0) % batch;
            if (slot == 0) {          // K1: SPO-VGL of the next `nb` electron steps, all walkers
                const int nb = min(batch, k0 + kn - k);
                int rc = spo_batch_vgl(d, sp, pos, delta + 3 * mv, k, nb,
                                       rec ? rec + mv / nw * (size_t)nrec * nel : nullptr, nrec, d->vgl, s);
                if (rc) return rc;
            }
            const float *phi = d->vgl + slot * slot_stride;
            // K2: ratio + row copy, K3: decision + rank-1 update
            prof_start(d, kProfRatio, s);
            QMC_WITH_B(d, TB, Bp, (ratio_rowcopy_kernel<TB><<<nw, 256, 0, s>>>(Bp, nel, d->ld, k, phi, (size_t)5 * d->np, d->np, d->rowk,
                                                                               d->ratio, force ? force + 3 * mv : nullptr)));
            prof_stop(d, s);
            QMC_LAUNCHED();
            UpdateArgs u{};
            u.B = d->b32 ? (void *)d->Bf : (void *)d->B; u.nel = nel; u.ld = d->ld; u.iel = k;
            u.phi = phi; u.ldphi = (size_t)5 * d->np; u.rowk = d->rowk;
            u.ratio = d->ratio;
            u.unif = unif + mv;
            u.forced = forced ? forced + mv : nullptr;
            u.fixed_node = fixed_node;
            u.ratios_out = ratios_out ? ratios_out + mv : nullptr;
            u.accept_out = accept_out ? accept_out + mv : nullptr;
            u.pos = pos; u.delta = delta + 3 * mv;
            u.logdet = d->logdet; u.sign = d->sign; u.naccept = d->naccept;
            prof_start(d, kProfUpdate, s);
            cudaError_t ue = d->b32 ? launch_sm_update<float, true>(u, nw, s) : launch_sm_update<double, true>(u, nw, s);
            prof_stop(d, s);
            QMC_CUDA(ue);
        }
    }
    return QMC_OK;
}

}  // namespace qmc

using namespace qmc;

extern "C" int qmc_sweep(qmc_det_t *d, const qmc_spline_t *sp, double *pos, const double *delta,
                         const double *unif, int nsweeps, double *ratios_out, unsigned char *accept_out,
                         const unsigned char *forced, void *stream)
{
    return sweep_impl(d, sp, pos, delta, unif, nsweeps, ratios_out, accept_out, forced, nullptr,
                      (cudaStream_t)stream);
}

extern "C" int qmc_sweep_ex(qmc_det_t *d, const qmc_spline_t *sp, double *pos, const double *delta,
                            const double *unif, int nsweeps, double *ratios_out, unsigned char *accept_out,
                            const unsigned char *forced, const qmc_sweep_opts_t *opts, void *stream)
{
    return sweep_impl(d, sp, pos, delta, unif, nsweeps, ratios_out, accept_out, forced, opts,
                      (cudaStream_t)stream);
}

extern "C" int qmc_sweep_host(qmc_det_t *d, const qmc_spline_t *sp, double *pos_h, const double *delta_h,
                              const double *unif_h, int nsweeps, double *ratios_h, unsigned char *accept_h,
                              void *stream)
{
    QMC_REQUIRE(d && sp && pos_h && delta_h && unif_h, "qmc_sweep_host: NULL argument");
    QMC_REQUIRE(nsweeps >= 0, "qmc_sweep_host: nsweeps=%d", nsweeps);
    cudaStream_t s = (cudaStream_t)stream;
    const size_t nw = d->nw, nel = d->nel, moves = (size_t)nsweeps * nel * nw;
    auto up = [](size_t b) { return (b + 255) / 256 * 256; };
    const size_t b_pos = up(nw * nel * 3 * sizeof(double)), b_delta = up(moves * 3 * sizeof(double));
    const size_t b_unif = up(moves * sizeof(double)), b_ratio = up(moves * sizeof(double)), b_acc = up(moves);
    const size_t total = b_pos + b_delta + b_unif + b_ratio + b_acc;
    if (d->stage_bytes < total) {
        QMC_CUDA(cudaStreamSynchronize(s));
        cudaFree(d->stage);
        d->stage = nullptr;
        d->stage_bytes = 0;
        cudaError_t e = cudaMalloc(&d->stage, total);
        if (e != cudaSuccess) {
            set_error("qmc_sweep_host: cudaMalloc(%zu bytes) -> %s", total, cudaGetErrorString(e));
            (void)cudaGetLastError();
            return QMC_ENOMEM;
        }
        d->stage_bytes = total;
    }
    char *base = (char *)d->stage;
    double *pos = (double *)base;
    double *delta = (double *)(base + b_pos);
    double *unif = (double *)(base + b_pos + b_delta);
    double *ratios = (double *)(base + b_pos + b_delta + b_unif);
    unsigned char *acc = (unsigned char *)(base + b_pos + b_delta + b_unif + b_ratio);
    QMC_CUDA(cudaMemcpyAsync(pos, pos_h, nw * nel * 3 * sizeof(double), cudaMemcpyHostToDevice, s));
    QMC_CUDA(cudaMemcpyAsync(delta, delta_h, moves * 3 * sizeof(double), cudaMemcpyHostToDevice, s));
    QMC_CUDA(cudaMemcpyAsync(unif, unif_h, moves * sizeof(double), cudaMemcpyHostToDevice, s));
    int rc = sweep_impl(d, sp, pos, delta, unif, nsweeps, ratios_h ? ratios : nullptr, accept_h ? acc : nullptr,
                        nullptr, nullptr, s);
    if (rc) return rc;
    QMC_CUDA(cudaMemcpyAsync(pos_h, pos, nw * nel * 3 * sizeof(double), cudaMemcpyDeviceToHost, s));
    if (ratios_h) QMC_CUDA(cudaMemcpyAsync(ratios_h, ratios, moves * sizeof(double), cudaMemcpyDeviceToHost, s));
    if (accept_h) QMC_CUDA(cudaMemcpyAsync(accept_h, acc, moves, cudaMemcpyDeviceToHost, s));
    QMC_CUDA(cudaStreamSynchronize(s));
    return QMC_OK;
}
