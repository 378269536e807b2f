// Delayed (rank-k) update of the inverse: "a delayed update algorithm that enables
// increased use of matrix-matrix multiplication [44]", L299.  The paper prints no formulas; these
// follow from the Woodbury identity on the definition (R:O7):
//
//   window: B0 = (A0^-1)^T is left untouched while up to K accepted moves (k_l, v_l), l < p, of
//   DISTINCT electrons are buffered.  S[l][m] = v_l . B0[k_m]  (p x p), kept as S^-1.
//   ratio of a proposal (k, v), k not in the window:
//       d = v . B0[k],  x_m = v . B0[k_m],  c_l = v_l . B0[k],   R = d - x^T S^-1 c
//   accept: append (k, v), save the row B0[k]; S^-1 grows by bordering with Schur complement R.
//   flush:  q_l(m) = v_l . B0[m] - [k_l == m],  t(m) = S^-1 q(m),
//           B[m] = B0[m] - sum_l t_l(m) * B0[k_l]      -- one pass over B: 16 N ld bytes / walker.
//
// This file is the STEP-BY-STEP form behind qmc_det_ratio / qmc_det_accept_update in delayed mode
// (one launch per call, 2p+1 dots against the window).  qmc_sweep uses the one-launch-per-window
// form in window.cu.  The host schedules the flushes, so no device -> host traffic is needed.
#include "delayed_device.cuh"
#include "spo_device.cuh"
#include "update_device.cuh"

namespace qmc {

constexpr int kStepThreads = 256;

struct DelayedStepArgs {
    const void *B;                // TB [nw][nel][ld]  (B0 during a window)
    int nel, ld, np, iel, K;
    const float *phi;             // [nw][ldphi]
    size_t ldphi;
    // window state
    int *win_count;               // [nw]
    int *win_iel;                 // [nw][K]
    float *win_phi;               // [nw][K][np]
    double *win_rows;             // [nw][K][ld]
    double *win_sinv;             // [nw][K][K]
    int *win_slot;                // [nw][K]  slot l of win_rows / win_phi holds accepted move l
    int mode;                     // 1 = ratio only, 2 = append only (the caller's decision)
    double *ratio_io;             // [nw]  mode 1: out
    const unsigned char *accept_in;   // [nw] mode 2
    double *logdet;
    int *sign;
    long long *naccept;
};

// One block per walker.  Each thread owns column quads j = 4*tid (+ 4*blockDim per pass): it
// accumulates the 2p+1 partial dots d, x_m, c_l over its columns; the block reduces them in a
// fixed order; warp 0 finishes the ratio and, on accept, the block grows the window (row copy,
// orbital vector copy, bordered S^-1).
template <typename TB, int KMAX>
__global__ void __launch_bounds__(kStepThreads) delayed_step_kernel(DelayedStepArgs a)
{
    constexpr int NV = 2 * KMAX + 1;
    __shared__ double s_part[NV][kStepThreads / 32];
    __shared__ double s_tot[NV];
    __shared__ double s_y[KMAX], s_z[KMAX];
    __shared__ int s_flag;
    const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int p = a.win_count[w];
    const int K = a.K, ld = a.ld, np = a.np;
    const TB *b0k = reinterpret_cast<const TB *>(a.B) + ((size_t)w * a.nel + a.iel) * ld;
    const float *phi = a.phi + (size_t)w * a.ldphi;
    const double *rows = a.win_rows + (size_t)w * K * ld;
    const float *vwin = a.win_phi + (size_t)w * K * np;

    double acc[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) acc[i] = 0.0;
    {
        for (int j = 4 * tid; j < np; j += 4 * kStepThreads) {
            const float4 f = *reinterpret_cast<const float4 *>(phi + j);
            const double2 ba = ld2(b0k + j);
            const double2 bb = ld2(b0k + j + 2);
            const double v0 = f.x, v1 = f.y, v2 = f.z, v3 = f.w;
            acc[0] = fma(v0, ba.x, fma(v1, ba.y, fma(v2, bb.x, fma(v3, bb.y, acc[0]))));
#pragma unroll
            for (int l = 0; l < KMAX; ++l) {
                if (l < p) {
                    const double2 ra = *reinterpret_cast<const double2 *>(rows + (size_t)l * ld + j);
                    const double2 rb = *reinterpret_cast<const double2 *>(rows + (size_t)l * ld + j + 2);
                    acc[1 + l] = fma(v0, ra.x, fma(v1, ra.y, fma(v2, rb.x, fma(v3, rb.y, acc[1 + l]))));
                    const float4 g = *reinterpret_cast<const float4 *>(vwin + (size_t)l * np + j);
                    acc[1 + KMAX + l] = fma((double)g.x, ba.x, fma((double)g.y, ba.y,
                                          fma((double)g.z, bb.x, fma((double)g.w, bb.y, acc[1 + KMAX + l]))));
                }
            }
        }
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            const bool live = (i == 0) || ((i - 1) % KMAX < p);
            if (live) {
                const double s = warp_sum(acc[i]);
                if (lane == 0) s_part[i][wid] = s;
            }
        }
    }
    __syncthreads();
    if (tid < NV) {
        const bool live = (tid == 0) || ((tid - 1) % KMAX < p);
        double s = 0.0;
        if (live)
            for (int q = 0; q < kStepThreads / 32; ++q) s += s_part[tid][q];
        s_tot[tid] = s;
    }
    __syncthreads();
    // d = s_tot[0], x_m = s_tot[1+m], c_l = s_tot[1+KMAX+l]
    const double *sinv = a.win_sinv + (size_t)w * K * K;
    if (tid < KMAX) {
        // y = S^-1 c, z = S^-T x  (needed for the ratio and for the bordering update)
        double y = 0.0, z = 0.0;
        if (tid < p)
            for (int m = 0; m < p; ++m) {
                y = fma(sinv[tid * K + m], s_tot[1 + KMAX + m], y);
                z = fma(sinv[m * K + tid], s_tot[1 + m], z);
            }
        s_y[tid] = y;
        s_z[tid] = z;
    }
    __syncthreads();
    if (tid == 0) {
        double R = s_tot[0];
        for (int m = 0; m < p; ++m) R -= s_tot[1 + m] * s_y[m];
        bool acc_w = false;
        if (a.mode == 2) acc_w = a.accept_in[w] != 0 && usable_ratio(R);   // the caller's decision (R equals the ratio it was given); R:A18
        else a.ratio_io[w] = R;
        s_tot[0] = R;
        s_flag = acc_w;
    }
    __syncthreads();
    if (a.mode == 1 || !s_flag) return;
    const double R = s_tot[0];
    if (tid == 0) {
        a.logdet[w] += log(fabs(R));
        if (R < 0.0) a.sign[w] = -a.sign[w];
        a.naccept[w] += 1;
        a.win_iel[(size_t)w * K + p] = a.iel;
        a.win_slot[(size_t)w * K + p] = p;
        a.win_count[w] = p + 1;
    }
    // append the orbital vector and the row B0[k]
    float *vdst = a.win_phi + ((size_t)w * K + p) * np;
    double *rdst = a.win_rows + ((size_t)w * K + p) * ld;
    for (int j = 4 * tid; j < np; j += 4 * kStepThreads)
        *reinterpret_cast<float4 *>(vdst + j) = *reinterpret_cast<const float4 *>(phi + j);
    for (int j = 2 * tid; j < ld; j += 2 * kStepThreads)
        *reinterpret_cast<double2 *>(rdst + j) = ld2(b0k + j);
    // bordered inverse: S'^-1 = [[S^-1 + y z^T / R, -y / R], [-z^T / R, 1 / R]]
    double *so = a.win_sinv + (size_t)w * K * K;
    const double rinv = 1.0 / R;
    for (int e = tid; e < (p + 1) * (p + 1); e += kStepThreads) {
        const int i = e / (p + 1), j = e % (p + 1);
        double val;
        if (i < p && j < p) val = so[i * K + j] + s_y[i] * s_z[j] * rinv;
        else if (i < p) val = -s_y[i] * rinv;
        else if (j < p) val = -s_z[j] * rinv;
        else val = rinv;
        so[i * K + j] = val;
    }
}

// The flush (two DMMA contractions in one pass over B) lives in flush.cu.

static cudaError_t launch_step(const DelayedStepArgs &a, int nw, int b32, cudaStream_t s)
{
    if (b32) {
        if (a.K <= 8) delayed_step_kernel<float, 8><<<nw, kStepThreads, 0, s>>>(a);
        else if (a.K <= 16) delayed_step_kernel<float, 16><<<nw, kStepThreads, 0, s>>>(a);
        else delayed_step_kernel<float, 32><<<nw, kStepThreads, 0, s>>>(a);
    } else {
        if (a.K <= 8) delayed_step_kernel<double, 8><<<nw, kStepThreads, 0, s>>>(a);
        else if (a.K <= 16) delayed_step_kernel<double, 16><<<nw, kStepThreads, 0, s>>>(a);
        else delayed_step_kernel<double, 32><<<nw, kStepThreads, 0, s>>>(a);
    }
    count_launch();
    return cudaGetLastError();
}

static void fill_common(DelayedStepArgs &a, qmc_det *d, int iel, const float *phi, size_t ldphi)
{
    a.B = d->b32 ? (const void *)d->Bf : (const void *)d->B;
    a.nel = d->nel; a.ld = d->ld; a.np = d->np; a.iel = iel; a.K = d->delay;
    a.phi = phi; a.ldphi = ldphi;
    a.win_count = d->win_count; a.win_iel = d->win_iel; a.win_slot = d->win_slot; a.win_phi = d->win_phi;
    a.win_rows = d->win_rows; a.win_sinv = d->win_sinv;
    a.logdet = d->logdet; a.sign = d->sign; a.naccept = d->naccept;
}

int delayed_ratio(qmc_det *d, int iel, const float *phi, int ldo, double *ratio, cudaStream_t s)
{
    QMC_REQUIRE(ldo >= d->np, "qmc_det_ratio (delayed): ldo=%d must be >= the table pitch %d", ldo, d->np);
    QMC_REQUIRE(ldo % 4 == 0 && ((uintptr_t)phi & 15) == 0, "qmc_det_ratio (delayed): phi must be 16-byte aligned with ldo %% 4 == 0 (ldo=%d)", ldo);
    // a second move of an electron already in the window would break row distinctness: flush first
    if (d->host_pending && d->win_host_iel[iel]) {
        int rc = delayed_flush_reset_host(d, s);
        if (rc) return rc;
    }
    DelayedStepArgs a{};
    fill_common(a, d, iel, phi, (size_t)ldo);
    a.mode = 1;
    a.ratio_io = ratio;
    prof_start(d, kProfDelayedRatio, s);
    cudaError_t e = launch_step(a, d->nw, d->b32, s);
    prof_stop(d, s);
    QMC_CUDA(e);
    return QMC_OK;
}

int delayed_accept(qmc_det *d, int iel, const float *phi, int ldo, const double *ratio,
                   const unsigned char *accept, cudaStream_t s)
{
    QMC_REQUIRE(ldo >= d->np, "qmc_det_accept_update (delayed): ldo=%d must be >= the table pitch %d", ldo, d->np);
    QMC_REQUIRE(ldo % 4 == 0 && ((uintptr_t)phi & 15) == 0, "qmc_det_accept_update (delayed): phi must be 16-byte aligned with ldo %% 4 == 0 (ldo=%d)", ldo);
    if (d->host_pending >= d->delay || (d->host_pending && d->win_host_iel[iel])) {
        int rc = delayed_flush_reset_host(d, s);
        if (rc) return rc;
    }
    DelayedStepArgs a{};
    fill_common(a, d, iel, phi, (size_t)ldo);
    a.mode = 2;
    (void)ratio;   // recomputed bit-identically from the same inputs
    a.accept_in = accept;
    prof_start(d, kProfDelayedAccept, s);
    cudaError_t e = launch_step(a, d->nw, d->b32, s);
    prof_stop(d, s);
    QMC_CUDA(e);
    d->host_pending += 1;
    d->win_host_iel[iel] = 1;
    d->win_rows_raw = 1;
    d->win_vec = d->win_phi;
    d->win_vec_wstride = (size_t)d->delay * d->np;
    d->win_vec_sstride = (size_t)d->np;
    return QMC_OK;
}

int delayed_flush_reset_host(qmc_det *d, cudaStream_t s)
{
    int rc = delayed_flush(d, s);
    if (rc) return rc;
    if (d->win_host_iel) memset(d->win_host_iel, 0, (size_t)d->nel);
    return QMC_OK;
}

}  // namespace qmc
