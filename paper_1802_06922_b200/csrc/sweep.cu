// qmc_sweep*: the particle-by-particle sweep driver (sec 5.2.1) -- all walkers
// in lockstep (L114, L181), electrons in sequence.  Launches:
//   K1 spo_batch_kernel      S0 proposal, S1 stencil, S2 SPO-VGL gather -- once per batch of steps
//   K2 ratio_rowcopy_kernel  S3 ratio, copy of row k                    -- per electron step
//   K3 sm_update_kernel      S4 Metropolis test, S5 rank-1 update       -- per electron step
// (delayed mode, per window of K steps: K1, then delayed_window_kernel = S3 + S4 of the K steps,
//  then flush_dmma_kernel = S5')
#include "delayed_device.cuh"
#include "jastrow_device.cuh"
#include "spo_device.cuh"
#include "update_device.cuh"

namespace qmc {

void spo_launch_shape(int np, int *threads, int *tiles);
int jastrow_move_launch(const qmc_jastrow *J, int nw, int nel, const double *pos, int nother, const double *other,
                        int iel0, int nb, const double *delta, const double *rnew, double *dj_out, double *ratio_out,
                        double *tfac_out, double *corr_out, int ncorr, cudaStream_t s, const int *cur = nullptr, int kend = 0);

__global__ void fill_int_kernel(int *p, int n, int v)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

// Jastrow factor of a sweep (qmc_sweep_opts_t.jastrow): what the step loops need.
struct SweepJastrow {
    const qmc_jastrow *J;     // NULL: none
    const double *other;
    int nother;
    double *jratio_out;       // [nsweeps][nel][nw] or NULL
};

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
    float *phi_record;     // [nb][nrecord][nel_record], offset to (sweep, first electron), or NULL
    int nrecord, nel_record;
    // QMC_DET_ACCEPT_WINDOWS: every walker is at its own electron; step j of the batch is electron cur[w] + j
    // (nothing to do beyond kend), delta and phi_record are then offset to (sweep, electron 0)
    // The SPO-VGL scratch is then a ring of `ring` slots (slot = electron % ring): only the proposals beyond
    // ev[w] (those the previous windows did not evaluate yet) are evaluated, up to cur[w] + nb.
    const int *cur, *ev;
    int kend, ring, nb;
};

// One block per (orbital tile, walker, step of the batch).  Thread t owns orbitals 4t..4t+3 of the
// tile: it gathers their value/gradient/Laplacian from the 64 stencil rows (S0-S2).
__global__ void __launch_bounds__(256) spo_batch_kernel(SpoBatchArgs a)
{
    __shared__ StencilSmem st;
    const int w = blockIdx.y, j = blockIdx.z;
    const int iel = a.cur ? a.ev[w] + j : a.iel0 + j;
    if (a.cur && iel >= min(a.cur[w] + a.nb, a.kend)) return;     // beyond this walker's next window (block-uniform)
    const int jd = a.cur ? iel : j;                        // index into delta / phi_record
    const int slot = a.cur ? iel % a.ring : j;             // where the result goes in the scratch
    const double *r = a.pos + ((size_t)w * a.nel + iel) * 3;
    double dx = 0.0, dy = 0.0, dz = 0.0;
    if (a.delta) {
        const double *dl = a.delta + 3 * ((size_t)jd * a.nw + w);
        dx = dl[0]; dy = dl[1]; dz = dl[2];
    }
    stage_stencil(a.sp, r[0] + dx, r[1] + dy, r[2] + dz, st);
    const int np = a.sp.np;
    const int col = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
    if (col >= np) return;
    float4 v, gx, gy, gz, lp;
    gather4<true>(a.sp, st, col, v, gx, gy, gz, lp);
    float *o = a.vgl + ((size_t)slot * a.nw + w) * 5 * np + col;
    *reinterpret_cast<float4 *>(o) = v;
    *reinterpret_cast<float4 *>(o + np) = gx;
    *reinterpret_cast<float4 *>(o + 2 * (size_t)np) = gy;
    *reinterpret_cast<float4 *>(o + 3 * (size_t)np) = gz;
    *reinterpret_cast<float4 *>(o + 4 * (size_t)np) = lp;
    if (a.phi_record && w < a.nrecord) {
        float *rec = a.phi_record + ((size_t)jd * a.nrecord + w) * a.nel_record;
        if (col + 0 < a.nel_record) rec[col + 0] = v.x;
        if (col + 1 < a.nel_record) rec[col + 1] = v.y;
        if (col + 2 < a.nel_record) rec[col + 2] = v.z;
        if (col + 3 < a.nel_record) rec[col + 3] = v.w;
    }
}

// S3 for the rank-1 path: R_w = B_w[iel] . phi_w (fp64, fixed order) and a copy of row iel, so that
// the update kernel can overwrite B in place.  One block per walker.  With force_out the three
// gradient vectors of the proposal (phi + np, + 2 np, + 3 np) are contracted with the same row:
// F = 2 grad log Psi_T at the proposed configuration = 2 (B[iel] . grad phi) / R.
// Drift moves (eq. 11-13; R:A20): what the ratio kernel needs to form the ratio of the
// transition densities, log T(r'->r)/T(r->r') = (|r' - r - tau F(r)|^2 - |r - r' - tau F(r')|^2) / (2 tau).
struct DriftStep {
    double tau;               // 0: no drift
    const double *pos;        // [nw][nel][3] current positions
    const double *rprop;      // [nw][3] proposed positions of this step
    const double *fcur;       // [nw][3] F_k(r) at the current configuration
    double *tfac;             // [nw] out: exp(log T ratio), the factor of eq. 12
    double *logt_out;         // [nw] out or NULL
};

// F_k(r) = 2 grad_k log|det A| = 2 sum_j grad phi_j(r_k) B[k][j] at the CURRENT configuration (L156) and
// the proposal of eq. 13 / eq. 19 with lambda = 1/2: r' = r_k + (tau F + chi), chi ~ N(0, tau) pre-generated.
// One block per walker; the three dots in a fixed order.
template <typename TB>
__global__ void __launch_bounds__(128)
drift_propose_kernel(const TB *__restrict__ B, int nel, int ld, int iel, const float *__restrict__ vgl_cur,
                     size_t ldv, int np, const double *__restrict__ pos, const double *__restrict__ chi,
                     double tau, double *__restrict__ rprop, double *__restrict__ fcur)
{
    __shared__ double red[33];
    const int w = blockIdx.x;
    const TB *row = B + ((size_t)w * nel + iel) * ld;
    const float *gv = vgl_cur + (size_t)w * ldv + np;          // d/dx, then d/dy, d/dz at + np each
    double g[3] = {0.0, 0.0, 0.0};
    for (int j = threadIdx.x; 2 * j < nel; j += 128) {         // the vectors are zero-padded up to np >= nel
        const double2 b = ld2(row + 2 * j);
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const float2 q = reinterpret_cast<const float2 *>(gv + (size_t)d * np)[j];
            g[d] = fma(b.x, (double)q.x, g[d]);
            g[d] = fma(b.y, (double)q.y, g[d]);
        }
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double f = 2.0 * block_sum(g[d], red);
        if (threadIdx.x == 0) {
            fcur[3 * (size_t)w + d] = f;
            // (no FMA contraction: the proposal is reproducible from fcur, chi and the position, bit for bit)
            rprop[3 * (size_t)w + d] = __dadd_rn(pos[((size_t)w * nel + iel) * 3 + d], __dadd_rn(__dmul_rn(tau, f), chi[3 * (size_t)w + d]));
        }
    }
}

template <typename TB>
__global__ void __launch_bounds__(256)
ratio_rowcopy_kernel(const TB *__restrict__ B, int nel, int ld, int iel, const float *__restrict__ phi,
                     size_t ldphi, int np, double *__restrict__ rowk, double *__restrict__ ratio,
                     double *__restrict__ force_out, DriftStep ds)
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
            if (force_out || ds.tau > 0.0) {
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
    if (force_out || ds.tau > 0.0) {
        double fnew[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double gd = block_sum(g[d], red);
            fnew[d] = acc != 0.0 ? 2.0 * gd / acc : 0.0;
            if (threadIdx.x == 0 && force_out) force_out[3 * (size_t)w + d] = fnew[d];
        }
        if (ds.tau > 0.0 && threadIdx.x == 0) {        // log T(r'->r)/T(r->r'), eq. 11-13 with lambda = 1/2
            double fwd = 0.0, bwd = 0.0;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const double rk = ds.pos[((size_t)w * nel + iel) * 3 + d], rn = ds.rprop[3 * (size_t)w + d];
                const double a = rn - rk - ds.tau * ds.fcur[3 * (size_t)w + d];
                const double b = rk - rn - ds.tau * fnew[d];
                fwd += a * a;
                bwd += b * b;
            }
            const double logt = (fwd - bwd) / (2.0 * ds.tau);
            ds.tfac[w] = exp(logt);
            if (ds.logt_out) ds.logt_out[w] = logt;
        }
    }
}

int spo_batch_vgl(qmc_det *d, const qmc_spline *sp, const double *pos, const double *delta, int iel0, int nb,
                  float *phi_record, int nrecord, float *out, cudaStream_t s, bool per_walker_cursor)
{
    int threads, tiles;
    spo_launch_shape(d->np, &threads, &tiles);
    SpoBatchArgs a{};
    a.sp = sp->view;
    a.pos = pos; a.delta = delta;
    a.nel = d->nel; a.iel0 = iel0; a.nw = d->nw;
    a.vgl = out;
    a.phi_record = phi_record; a.nrecord = nrecord; a.nel_record = d->nel;
    if (per_walker_cursor) { a.cur = d->cur; a.ev = d->cur + d->nw; a.kend = d->win_kend; a.ring = d->vgl_ring; a.nb = nb; }
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
                         const SweepJastrow &jas, cudaStream_t s)
{
    const int nw = d->nw, nel = d->nel, batch = d->spo_batch;
    const bool aw = d->accept_windows != 0;
    // accept windows: a window takes at least min(delay, remaining) steps of every walker, so ceil(kn / delay)
    // windows always finish the sweep (the last ones find most walkers done: their CTAs exit at once)
    const int wins_per_sweep = aw ? (kn + d->delay - 1) / d->delay : (kn + batch - 1) / batch;
    if (aw) d->win_kend = k0 + kn;
    const long long nwin = (long long)nsweeps * wins_per_sweep;
    if (nwin == 0) return QMC_OK;
    bool overlap = d->overlap && !d->prof_on;     // per-kernel event timing needs the kernels one after another
    auto vbuf = [&](long long i) { return d->vgl_buf[(overlap && !aw) ? (i & 1) : 0]; };   // accept windows: one ring
    if (overlap && !d->aux) {
        QMC_CUDA(cudaStreamCreateWithFlags(&d->aux, cudaStreamNonBlocking));
        QMC_CUDA(cudaEventCreateWithFlags(&d->ev_spo[0], cudaEventDisableTiming));
        QMC_CUDA(cudaEventCreateWithFlags(&d->ev_spo[1], cudaEventDisableTiming));
        QMC_CUDA(cudaEventCreateWithFlags(&d->ev_main, cudaEventDisableTiming));
    }
    auto spo = [&](long long i, cudaStream_t st) -> int {     // K1 of window i into buffer i & 1
        const int sw = (int)(i / wins_per_sweep);
        if (aw) {                                             // every walker from its own cursor; arrays offset to the sweep
            const size_t mv0 = (size_t)sw * nel * nw;
            return spo_batch_vgl(d, sp, pos, delta + 3 * mv0, 0, batch, rec ? rec + mv0 / nw * (size_t)nrec * nel : nullptr,
                                 nrec, vbuf(i), st, true);
        }
        const int k = k0 + (int)(i % wins_per_sweep) * batch;
        const int nb = min(batch, k0 + kn - k);
        const size_t mv = ((size_t)sw * nel + k) * nw;
        return spo_batch_vgl(d, sp, pos, delta + 3 * mv, k, nb, rec ? rec + mv / nw * (size_t)nrec * nel : nullptr,
                             nrec, vbuf(i), st, false);
    };
    auto reset_cursors = [&]() -> int {                       // start of a sweep: every walker at electron k0
        fill_int_kernel<<<(2 * nw + 127) / 128, 128, 0, s>>>(d->cur, 2 * nw, k0);      // cursors and evaluated-up-to marks
        QMC_LAUNCHED();
        return QMC_OK;
    };
    int rc;
    if (aw && (rc = reset_cursors())) return rc;
    if (overlap) {
        QMC_CUDA(cudaEventRecord(d->ev_main, s));
        QMC_CUDA(cudaStreamWaitEvent(d->aux, d->ev_main, 0));
        if ((rc = spo(0, d->aux))) return rc;
        QMC_CUDA(cudaEventRecord(d->ev_spo[0], d->aux));
    }
    for (long long i = 0; i < nwin; ++i) {
        const int sw = (int)(i / wins_per_sweep);
        // accept windows: the per-move arrays are offset to the sweep and indexed with the walker's own electron
        const int k = aw ? 0 : k0 + (int)(i % wins_per_sweep) * batch;
        const int nb = aw ? batch : min(batch, k0 + kn - k);
        const size_t mv = ((size_t)sw * nel + k) * nw;
        if (overlap) QMC_CUDA(cudaStreamWaitEvent(s, d->ev_spo[i & 1], 0));
        else if ((rc = spo(i, s))) return rc;
        d->vgl = vbuf(i);
        WindowJastrow wj{};
        if (jas.J) {
            // dJ of the window's nb proposals against the configuration at the start of the window, and for every
            // pair of steps m < j what an accepted move m changes in dJ of step j; the window kernel adds the
            // pair terms of the steps it has accepted by then
            double *corr = d->jas_dj + (size_t)batch * nw;
            if ((rc = jastrow_move_launch(jas.J, nw, nel, pos, jas.nother, jas.other, k, nb, delta + 3 * mv, nullptr,
                                          d->jas_dj, nullptr, nullptr, corr, batch, s, aw ? d->cur : nullptr, d->win_kend))) return rc;
            wj.base = d->jas_dj; wj.corr = corr; wj.ncorr = batch; wj.jratio_out = jas.jratio_out ? jas.jratio_out + mv : nullptr;
        }
        rc = delayed_sweep_window(d, pos, delta + 3 * mv, unif + mv, k, nb, ratios_out ? ratios_out + mv : nullptr,
                                  accept_out ? accept_out + mv : nullptr, forced ? forced + mv : nullptr, fixed_node,
                                  force ? force + 3 * mv : nullptr, overlap && i + 1 < nwin ? 1 : 0, wj, s);
        if (rc) return rc;
        if (aw && i + 1 < nwin && (i + 1) % wins_per_sweep == 0) {
            // next window starts a new sweep: cursors back to k0 (after this window's kernel, before the next SPO)
            if ((rc = reset_cursors())) return rc;
            if (overlap) QMC_CUDA(cudaEventRecord(d->ev_main, s));
        }
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

// Drift moves (R:A20).  The proposal of electron k now depends on the decisions
// before it (F_k(r) is taken with the current inverse), so per electron step:
//   D1 drift_propose_kernel  F_k(r) from the gradients at the CURRENT position, r' = r + tau F + chi
//   D2 spo_batch_kernel      SPO-VGL at r' (one position per walker)
//   D3 ratio_rowcopy_kernel  R, F_k(r') and the factor T(r'->r)/T(r->r') of eq. 12
//   D4 sm_update_kernel      accept iff R^2 T'/T > u; rank-1 update
// and once per 16 electrons a batched SPO-VGL at their current positions (those do not change until the
// electron's own step), which is what survives of the batched gather.  delay_rank >= 2 is served by
// the same per-step kernels after the pending window has been applied (every step is then a rank-1
// update: the one-launch-per-window form needs all proposals of a window up front).
static int sweep_drift(qmc_det *d, const qmc_spline *sp, double *pos, const double *chi, const double *unif,
                       int nsweeps, int k0, int kn, double *ratios_out, unsigned char *accept_out,
                       const unsigned char *forced, int fixed_node, double *force, float *rec, int nrec, double tau,
                       double *rprop_out, double *logt_out, double *fcur_out, cudaStream_t s)
{
    const int nw = d->nw, nel = d->nel, np = d->np;
    if (d->delay) {
        int rc = delayed_flush_reset_host(d, s);
        if (rc) return rc;
    }
    if (!d->vgl_cur) {
        auto alloc = [&](void **p, size_t bytes) {
            cudaError_t e = cudaMalloc(p, bytes);
            if (e != cudaSuccess) { set_error("qmc_sweep_ex (drift): cudaMalloc(%zu bytes) -> %s", bytes, cudaGetErrorString(e)); (void)cudaGetLastError(); return QMC_ENOMEM; }
            return QMC_OK;
        };
        int rc;
        if ((rc = alloc((void **)&d->vgl_cur, (size_t)kSpoBatch * nw * 5 * np * sizeof(float))) ||
            (rc = alloc((void **)&d->rprop, (size_t)nw * 3 * sizeof(double))) ||
            (rc = alloc((void **)&d->fcur, (size_t)nw * 3 * sizeof(double))) ||
            (rc = alloc((void **)&d->tfac, (size_t)nw * sizeof(double)))) return rc;
    }
    int threads, tiles;
    spo_launch_shape(np, &threads, &tiles);
    const size_t slot_stride = (size_t)nw * 5 * np;
    float *const vgl_prop = d->vgl_buf[0];                 // slot 0 of the proposal scratch
    for (int sw = 0; sw < nsweeps; ++sw) {
        for (int k = k0; k < k0 + kn; ++k) {
            const size_t mv = ((size_t)sw * nel + k) * nw;
            const int slot = (k - k0) % kSpoBatch;
            if (slot == 0) {          // gradients at the current positions of the next 16 electrons
                const int nb = min(kSpoBatch, k0 + kn - k);
                int rc = spo_batch_vgl(d, sp, pos, nullptr, k, nb, nullptr, 0, d->vgl_cur, s, false);
                if (rc) return rc;
            }
            double *rprop = rprop_out ? rprop_out + 3 * mv : d->rprop;
            double *fcur = fcur_out ? fcur_out + 3 * mv : d->fcur;
            prof_start(d, kProfRatio, s);
            QMC_WITH_B(d, TB, Bp, (drift_propose_kernel<TB><<<nw, 128, 0, s>>>(Bp, nel, d->ld, k, d->vgl_cur + slot * slot_stride,
                                                                               (size_t)5 * np, np, pos, chi + 3 * mv, tau, rprop, fcur)));
            prof_stop(d, s);
            QMC_LAUNCHED();
            SpoBatchArgs a{};         // D2: one position per walker, read from rprop ([nw][1][3])
            a.sp = sp->view; a.pos = rprop; a.delta = nullptr; a.nel = 1; a.iel0 = 0; a.nw = nw;
            a.vgl = vgl_prop;
            a.phi_record = rec ? rec + mv / nw * (size_t)nrec * nel : nullptr; a.nrecord = nrec; a.nel_record = nel;
            prof_start(d, kProfSpoRatio, s);
            spo_batch_kernel<<<dim3(tiles, nw, 1), threads, 0, s>>>(a);
            prof_stop(d, s);
            QMC_LAUNCHED();
            DriftStep ds{tau, pos, rprop, fcur, d->tfac, logt_out ? logt_out + mv : nullptr};
            prof_start(d, kProfRatio, s);
            QMC_WITH_B(d, TB, Bp, (ratio_rowcopy_kernel<TB><<<nw, 256, 0, s>>>(Bp, nel, d->ld, k, vgl_prop, (size_t)5 * np, np, d->rowk,
                                                                               d->ratio, force ? force + 3 * mv : nullptr, ds)));
            prof_stop(d, s);
            QMC_LAUNCHED();
            UpdateArgs u{};
            u.B = d->b32 ? (void *)d->Bf : (void *)d->B; u.nel = nel; u.ld = d->ld; u.iel = k;
            u.phi = vgl_prop; u.ldphi = (size_t)5 * np; u.rowk = d->rowk;
            u.ratio = d->ratio; u.tfac = d->tfac; u.rprop = rprop;
            u.unif = unif + mv;
            u.forced = forced ? forced + mv : nullptr;
            u.fixed_node = fixed_node;
            u.ratios_out = ratios_out ? ratios_out + mv : nullptr;
            u.accept_out = accept_out ? accept_out + mv : nullptr;
            u.pos = pos; u.delta = chi + 3 * mv;
            u.logdet = d->logdet; u.sign = d->sign; u.naccept = d->naccept;
            prof_start(d, kProfUpdate, s);
            cudaError_t ue = d->b32 ? launch_sm_update<float, true>(u, nw, s) : launch_sm_update<double, true>(u, nw, s);
            prof_stop(d, s);
            QMC_CUDA(ue);
        }
    }
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
        QMC_REQUIRE(opts->drift_tau >= 0.0 && isfinite(opts->drift_tau), "qmc_sweep_ex: drift_tau=%g", opts->drift_tau);
        QMC_REQUIRE(!(opts->jastrow && opts->drift_tau > 0.0), "qmc_sweep_ex: a Jastrow factor with drift moves needs grad J, which is not built");
        if (opts->drift_tau > 0.0)
            return sweep_drift(d, sp, pos, delta, unif, nsweeps, k0, kn, ratios_out, accept_out, forced, fixed_node, force,
                               rec, nrec, opts->drift_tau, opts->rprop_out, opts->logt_out, opts->fcur_out, s);
    }
    const int batch = d->spo_batch;
    const size_t slot_stride = (size_t)nw * 5 * d->np;
    SweepJastrow jas{};
    if (opts && opts->jastrow) {
        jas.J = opts->jastrow;
        jas.nother = opts->jastrow_nother;
        jas.other = jas.nother > 0 ? opts->jastrow_other : nullptr;
        jas.jratio_out = opts->jratio_out;
        QMC_REQUIRE(jas.nother >= 0 && (jas.nother == 0 || jas.other), "qmc_sweep_ex: jastrow_nother=%d without positions", jas.nother);
        QMC_REQUIRE(jas.J->device == d->device, "qmc_sweep_ex: the Jastrow factor lives on another device");
        if (!d->jas_dj) {
            const size_t kk = d->delay > 1 ? d->spo_batch : 1;   // dJ [K][nw] + pair terms [nw][K][K], K = steps per window
            const size_t bytes = (kk * nw + (size_t)nw * kk * kk) * sizeof(double);
            cudaError_t e = cudaMalloc((void **)&d->jas_dj, bytes);
            if (e != cudaSuccess) { set_error("qmc_sweep_ex (jastrow): cudaMalloc(%zu bytes) -> %s", bytes, cudaGetErrorString(e)); (void)cudaGetLastError(); return QMC_ENOMEM; }
        }
    }
    if (d->delay) return sweep_delayed(d, sp, pos, delta, unif, nsweeps, k0, kn, ratios_out, accept_out, forced,
                                       fixed_node, force, rec, nrec, jas, s);
    for (int sw = 0; sw < nsweeps; ++sw) {
        for (int k = k0; k < k0 + kn; ++k) {
            const size_t mv = ((size_t)sw * nel + k) * nw;
            const int slot = (k - k0) % batch;
            if (slot == 0) {          // K1: SPO-VGL of the next `nb` electron steps, all walkers
                const int nb = min(batch, k0 + kn - k);
                int rc = spo_batch_vgl(d, sp, pos, delta + 3 * mv, k, nb,
                                       rec ? rec + mv / nw * (size_t)nrec * nel : nullptr, nrec, d->vgl, s, false);
                if (rc) return rc;
            }
            const float *phi = d->vgl + slot * slot_stride;
            // K2: ratio + row copy, K3: decision + rank-1 update
            prof_start(d, kProfRatio, s);
            QMC_WITH_B(d, TB, Bp, (ratio_rowcopy_kernel<TB><<<nw, 256, 0, s>>>(Bp, nel, d->ld, k, phi, (size_t)5 * d->np, d->np, d->rowk,
                                                                               d->ratio, force ? force + 3 * mv : nullptr, DriftStep{})));
            prof_stop(d, s);
            QMC_LAUNCHED();
            UpdateArgs u{};
            u.B = d->b32 ? (void *)d->Bf : (void *)d->B; u.nel = nel; u.ld = d->ld; u.iel = k;
            u.phi = phi; u.ldphi = (size_t)5 * d->np; u.rowk = d->rowk;
            u.ratio = d->ratio;
            if (jas.J) {              // exp(-2 dJ) at the current configuration: the Jastrow part of |Psi'/Psi|^2
                int rc = jastrow_move_launch(jas.J, nw, nel, pos, jas.nother, jas.other, k, 1, delta + 3 * mv, nullptr, nullptr,
                                             jas.jratio_out ? jas.jratio_out + mv : nullptr, d->jas_dj, nullptr, 0, s);
                if (rc) return rc;
                u.tfac = d->jas_dj;
            }
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
