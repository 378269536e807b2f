// One WINDOW of the delayed (rank-k) update inside qmc_sweep: the K consecutive electron steps
// k0 .. k0+nb-1 of the lockstep sweep in ONE launch (DESIGN.md R:O7, R:A14).
//
// Every quantity the nb sequential ratios and decisions need is an entry of one small matrix:
// the proposals of the window are known up front (r' = pos[w][k] + delta does not depend on the
// outcome of earlier moves of OTHER electrons, and their orbital vectors v_i come from the batched
// SPO-VGL launch), and every row of B0 the window touches is one of B0[k0 .. k0+nb-1].  With
//
//     G[i][j] = v_i . B0[k0+j]                 (nb x nb, one (nb x N)(N x nb) fp64 contraction)
//
// the ratio of step i against the accepted steps l_0 < l_1 < ... < l_{p-1} < i is
//
//     d = G[i][i],   x_m = G[i][l_m],   c_m = G[l_m][i],   R = d - x^T S^-1 c,   S[a][b] = G[l_a][l_b]
//
// so the steps are O(p^2) scalar work on S^-1 (grown by bordering), done by one warp with no
// further pass over B0 or the vectors.  The kernel then leaves what the flush kernel consumes:
// count, electron indices, slots (= step index in the window, where the flush finds v_l) and
// R' = S^-T Rows (Rows[l] = B0[k_l]; the flush overwrites B in place and computes B -= Q R').
#include "delayed_device.cuh"
#include "dmma.cuh"
#include "update_device.cuh"

namespace qmc {

constexpr int kWinThreads = 256;

struct WindowArgs {
    const void *B;                // TB [nw][nel][ld]  B0 of the window
    int nw, nel, ld, np, K;
    int iel0, nb;                 // electrons iel0 .. iel0+nb-1, nb <= K
    const float *vgl;             // [nb][nw][5][np] SPO-VGL of the window's proposals (values first)
    const double *unif;           // [nb][nw]
    const unsigned char *forced;  // [nb][nw] or NULL
    int fixed_node;               // reject R < 0
    double *force_out;            // [nb][nw][3] or NULL: F = 2 grad log Psi_T at the proposed configuration
    double *ratios_out;           // [nb][nw] or NULL
    unsigned char *accept_out;    // [nb][nw] or NULL
    double *pos;                  // [nw][nel][3]
    const double *delta;          // [nb][nw][3]
    double *logdet;
    int *sign;
    long long *naccept;
    int *win_count;               // [nw]
    int *win_iel;                 // [nw][K]
    int *win_slot;                // [nw][K]
    double *win_rows;             // [nw][K][ld]   row l <- R'[l]
    WindowJastrow jas;            // base == NULL: no Jastrow factor
    // QMC_DET_ACCEPT_WINDOWS: the walker's window starts at electron cur[w], ends before kend, and closes when
    // pmax moves have been accepted; the per-move arrays are then offset to (sweep, electron 0)
    int *cur, *ev;                // ev[w]: electron up to which the walker's proposals have been evaluated
    int kend, pmax, ring;         // ring: slots of the SPO-VGL scratch (slot = electron % ring); 0: slot = step
};

// G[i][j] = x_i . B0[iel0 + j] for the nb vectors x_i = x0 + i * vstep (fp32) of one walker, into
// shared memory: warp q contracts the 16-column chunks q, q+8, ... with DMMA.8x8x4 (the contraction
// index inside a chunk is permuted so that one lane's float4 / 2 x double2 serve four k-steps), then
// the 8 partial G are summed in a fixed order.  Ends with a __syncthreads().
template <int KMAX, typename TB>
__device__ __forceinline__ void window_contract(const float *x0, size_t vstep, const TB *b0, int nb, int ld,
                                                int np, double *G_dst, int slot0, int ring)
{
    constexpr int MB = KMAX / 8;
    constexpr int GS = KMAX + 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    double acc[MB][MB][2];
#pragma unroll
    for (int i = 0; i < MB; ++i)
#pragma unroll
        for (int j = 0; j < MB; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const float *xrow[MB];                                 // vector of step 8 ib + g (ring: slot = electron % ring)
#pragma unroll
    for (int ib = 0; ib < MB; ++ib) {
        const int i = 8 * ib + g;
        xrow[ib] = x0 + (size_t)(ring ? (slot0 + i) % ring : i) * vstep;
    }
    for (int c0 = 16 * warp; c0 < np; c0 += 16 * (kWinThreads / 32)) {
        const int col = c0 + 4 * t;
        double av[MB][4], bv[MB][4];
#pragma unroll
        for (int jb = 0; jb < MB; ++jb) {
            const int j = 8 * jb + g;
            double2 lo = make_double2(0.0, 0.0), hi = lo;
            if (j < nb) {
                lo = ld2(b0 + (size_t)j * ld + col);
                hi = ld2(b0 + (size_t)j * ld + col + 2);
            }
            bv[jb][0] = lo.x; bv[jb][1] = lo.y; bv[jb][2] = hi.x; bv[jb][3] = hi.y;
        }
#pragma unroll
        for (int ib = 0; ib < MB; ++ib) {
            const int i = 8 * ib + g;
            float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
            if (i < nb) f = *reinterpret_cast<const float4 *>(xrow[ib] + col);
            av[ib][0] = f.x; av[ib][1] = f.y; av[ib][2] = f.z; av[ib][3] = f.w;
        }
#pragma unroll
        for (int s = 0; s < 4; ++s)
#pragma unroll
            for (int ib = 0; ib < MB; ++ib)
#pragma unroll
                for (int jb = 0; jb < MB; ++jb)
                    if (8 * ib < nb && 8 * jb < nb) dmma884(acc[ib][jb][0], acc[ib][jb][1], av[ib][s], bv[jb][s]);
    }
    for (int q = 0; q < kWinThreads / 32; ++q) {
        if (warp == q) {
#pragma unroll
            for (int ib = 0; ib < MB; ++ib)
#pragma unroll
                for (int jb = 0; jb < MB; ++jb) {
                    double *dst = G_dst + (8 * ib + g) * GS + 8 * jb + 2 * t;
                    if (q == 0) { dst[0] = acc[ib][jb][0]; dst[1] = acc[ib][jb][1]; }
                    else { dst[0] += acc[ib][jb][0]; dst[1] += acc[ib][jb][1]; }
                }
        }
        __syncthreads();
    }
}

// The same G for windows of more than 16 steps, where the KMAX/8 x KMAX/8 accumulator blocks of
// window_contract no longer fit a 64-register budget: warp (jb, part) owns the 8 columns 8 jb .. 8 jb + 7
// of G (the rows B0[iel0 + 8 jb ..]) and contracts the 16-column chunks part, part + NPART, ...; every row
// of B0 is still read once per block (the fp32 vectors are re-read by the KMAX/8 column blocks: L1 hits),
// and the NPART partial sums of a column block are added in a fixed order.  Ends with a __syncthreads().
template <int KMAX, typename TB>
__device__ __forceinline__ void window_contract_split(const float *x0, size_t vstep, const TB *b0, int nb, int ld,
                                                      int np, double *G_dst, int slot0, int ring)
{
    constexpr int MB = KMAX / 8;
    constexpr int GS = KMAX + 1;
    constexpr int NPART = (kWinThreads / 32) / MB;        // warps per column block (warps beyond MB * NPART idle)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int jb = warp / NPART, part = warp % NPART;
    double acc[MB][2];
#pragma unroll
    for (int i = 0; i < MB; ++i) acc[i][0] = acc[i][1] = 0.0;
    if (jb < MB && 8 * jb < nb) {
        const float *xrow[MB];
#pragma unroll
        for (int ib = 0; ib < MB; ++ib) {
            const int i = 8 * ib + g;
            xrow[ib] = x0 + (size_t)(ring ? (slot0 + i) % ring : i) * vstep;
        }
        const int j = 8 * jb + g;
        const TB *brow = b0 + (size_t)j * ld;
        for (int c0 = 16 * part; c0 < np; c0 += 16 * NPART) {
            const int col = c0 + 4 * t;
            double2 lo = make_double2(0.0, 0.0), hi = lo;
            if (j < nb) {
                lo = ld2(brow + col);
                hi = ld2(brow + col + 2);
            }
            const double bv[4] = {lo.x, lo.y, hi.x, hi.y};
            double av[MB][4];
#pragma unroll
            for (int ib = 0; ib < MB; ++ib) {
                float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
                if (8 * ib + g < nb) f = *reinterpret_cast<const float4 *>(xrow[ib] + col);
                av[ib][0] = f.x; av[ib][1] = f.y; av[ib][2] = f.z; av[ib][3] = f.w;
            }
#pragma unroll
            for (int s = 0; s < 4; ++s)
#pragma unroll
                for (int ib = 0; ib < MB; ++ib)
                    if (8 * ib < nb) dmma884(acc[ib][0], acc[ib][1], av[ib][s], bv[s]);
        }
    }
    for (int q = 0; q < NPART; ++q) {
        if (jb < MB && part == q) {
#pragma unroll
            for (int ib = 0; ib < MB; ++ib) {
                double *dst = G_dst + (8 * ib + g) * GS + 8 * jb + 2 * t;
                if (q == 0) { dst[0] = acc[ib][0]; dst[1] = acc[ib][1]; }
                else { dst[0] += acc[ib][0]; dst[1] += acc[ib][1]; }
            }
        }
        __syncthreads();
    }
}

template <int KMAX, typename TB>
__device__ __forceinline__ void window_G(const float *x0, size_t vstep, const TB *b0, int nb, int ld, int np,
                                         double *G_dst, int slot0, int ring)
{
    if (KMAX > 16) window_contract_split<KMAX, TB>(x0, vstep, b0, nb, ld, np, G_dst, slot0, ring);
    else window_contract<KMAX, TB>(x0, vstep, b0, nb, ld, np, G_dst, slot0, ring);
}

// One block per walker, 8 warps.  Phases 1-2: G (and, with FORCE, the same contraction for the three
// gradient vectors of every proposal).  Phase 3: warp 0 walks the nb steps.  Phase 4: R' = S^-T Rows,
// 8-column tiles over the warps.  KMAX bounds the steps of a window, PMAX <= KMAX the moves it can accept
// (accept windows: 24 proposals, 16 accepts), which is what sizes the registers of phase 4.
template <typename TB, int KMAX, bool FORCE, bool JAS, int PMAX = KMAX>
__global__ void __launch_bounds__(kWinThreads, (FORCE || KMAX > 24) ? 1 : ((KMAX > 16 && PMAX > 16) ? 2 : 4))
delayed_window_kernel(WindowArgs a)
{
    constexpr int GS = KMAX + 1;
    __shared__ double G_s[KMAX * GS];
    __shared__ double Gd_s[FORCE ? 3 * KMAX * GS : 1];     // Gd[d][i][j] = d_d phi(r'_i) . B0[iel0 + j]
    __shared__ double sinv_s[KMAX * GS];
    __shared__ long long rowoff_s[KMAX];
    __shared__ int p_s;
    const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int iel0 = a.cur ? a.cur[w] : a.iel0;            // first electron of this walker's window
    const int ebase = a.cur ? iel0 : 0;                    // index of step 0 in the per-move arrays
    const int nb = a.cur ? min(a.nb, a.kend - iel0) : a.nb;
    const int ld = a.ld, np = a.np, K = a.K;
    if (nb <= 0) {                                         // this walker has finished its sweep (block-uniform)
        if (tid == 0) a.win_count[w] = 0;
        return;
    }
    const size_t vstep = (size_t)a.nw * 5 * np;             // stride between steps in vgl
    const float *v0 = a.vgl + (size_t)w * 5 * np;
    const TB *b0 = reinterpret_cast<const TB *>(a.B) + ((size_t)w * a.nel + iel0) * ld;

    const int ring = a.cur ? a.ring : 0;
    window_G<KMAX, TB>(v0, vstep, b0, nb, ld, np, G_s, iel0, ring);
    if (FORCE)
        for (int d = 0; d < 3; ++d) window_G<KMAX, TB>(v0 + (size_t)(1 + d) * np, vstep, b0, nb, ld, np, Gd_s + d * KMAX * GS, iel0, ring);

    // ---- phase 3: the nb steps in sequence; lane m owns accepted move m (its step index `mine`).
    // Everything that lives in global memory stays outside the sequential loop: lane i fetches the
    // uniform / forced decision of step i before it and writes ratio, decision and the moved
    // position of step i after it, so a step costs shuffles, shared memory and fp64 arithmetic only.
    if (warp == 0) {
        const size_t mv_l = (size_t)(ebase + lane) * a.nw + w;        // move of step `lane`
        const bool step_l = lane < nb;
        const double u_l = (step_l && !a.forced) ? a.unif[mv_l] : 0.0;
        const int f_l = (step_l && a.forced) ? (a.forced[mv_l] != 0) : 0;
        double R_l = 1.0;                                             // ratio of step `lane`
        double F_l[3] = {0.0, 0.0, 0.0};                              // force of step `lane`
        // Jastrow factor: lane l holds dJ of step l against the window-start configuration
        constexpr bool jas = JAS;
        double dj_l = 0.0, jr_l = 1.0;
        if (jas && step_l) dj_l = a.jas.base[(size_t)lane * a.nw + w];
        const double *corr_w = jas ? a.jas.corr + (size_t)w * a.jas.ncorr * a.jas.ncorr : nullptr;
        unsigned acc_mask = 0;                                        // accepted steps (same in every lane)
        int p = 0, mine = 0;
        int nproc = nb;                                               // steps this window really takes
        for (int i = 0; i < nb; ++i) {
            if (p == a.pmax) { nproc = i; break; }                    // the window is full (accept windows; warp-uniform)
            const double c = lane < p ? G_s[mine * GS + i] : 0.0;     // c_m = v_{l_m} . B0[k_i]
            const double x = lane < p ? G_s[i * GS + mine] : 0.0;     // x_m = v_i . B0[k_{l_m}]
            double y = 0.0, z = 0.0;                                  // y = S^-1 c, z = S^-T x
            for (int q = 0; q < p; ++q) {
                const double cq = __shfl_sync(0xffffffffu, c, q), xq = __shfl_sync(0xffffffffu, x, q);
                if (lane < p) {
                    y = fma(sinv_s[lane * GS + q], cq, y);
                    z = fma(sinv_s[q * GS + lane], xq, z);
                }
            }
            const double R = G_s[i * GS + i] - warp_sum(x * y);
            const double u_i = __shfl_sync(0xffffffffu, u_l, i);
            const int f_i = __shfl_sync(0xffffffffu, f_l, i);
            double tf = 1.0;                                          // exp(-2 dJ): the Jastrow part of |Psi'/Psi|^2
            if (jas) {
                // the electrons of the accepted steps m < i sit at their proposed positions now: add their pair
                // terms (lane m owns step m; fixed butterfly order)
                const double corr = (lane < i && ((acc_mask >> lane) & 1u)) ? corr_w[(size_t)i * a.jas.ncorr + lane] : 0.0;
                const double dj = __shfl_sync(0xffffffffu, dj_l, i) + warp_sum(corr);
                tf = exp(-2.0 * dj);
                if (lane == i) jr_l = exp(-dj);
            }
            const bool acc_w = (a.forced ? (f_i != 0) : (metropolis_t(R, tf, u_i) && !(a.fixed_node && R < 0.0))) && usable_ratio(R);
            if (lane == i) R_l = R;
            if (FORCE) {
                // grad phi(r'_i) . B_cur[k_i] = gd - xg^T S^-1 c with the same y = S^-1 c as the ratio
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const double *Gd = Gd_s + d * KMAX * GS;
                    const double xg = lane < p ? Gd[i * GS + mine] : 0.0;
                    const double gd = Gd[i * GS + i] - warp_sum(xg * y);
                    if (lane == i) F_l[d] = R != 0.0 ? 2.0 * gd / R : 0.0;
                }
            }
            if (!acc_w) continue;
            acc_mask |= 1u << i;
            const double rinv = 1.0 / R;
            __syncwarp();             // every lane has read the old S^-1
            // bordered inverse: S'^-1 = [[S^-1 + y z^T / R, -y / R], [-z^T / R, 1 / R]]
            for (int q = 0; q < p; ++q) {
                const double zq = __shfl_sync(0xffffffffu, z, q);
                if (lane < p) sinv_s[lane * GS + q] += y * zq * rinv;
            }
            if (lane < p) {
                sinv_s[lane * GS + p] = -y * rinv;
                sinv_s[p * GS + lane] = -z * rinv;
            }
            if (lane == p) { sinv_s[p * GS + p] = rinv; mine = i; }
            ++p;
            __syncwarp();
        }
        // results of step `lane` (only the steps the window took)
        const bool done_l = lane < nproc;
        const bool acc_l = done_l && ((acc_mask >> lane) & 1u);
        if (done_l) {
            if (a.ratios_out) a.ratios_out[mv_l] = R_l;
            if (a.accept_out) a.accept_out[mv_l] = acc_l ? 1 : 0;
            if (jas && a.jas.jratio_out) a.jas.jratio_out[mv_l] = jr_l;
            if (FORCE) {
                a.force_out[3 * mv_l + 0] = F_l[0];
                a.force_out[3 * mv_l + 1] = F_l[1];
                a.force_out[3 * mv_l + 2] = F_l[2];
            }
        }
        if (acc_l) {
            double *r = a.pos + ((size_t)w * a.nel + iel0 + lane) * 3;
            r[0] += a.delta[3 * mv_l + 0];
            r[1] += a.delta[3 * mv_l + 1];
            r[2] += a.delta[3 * mv_l + 2];
        }
        const double logdet_add = warp_sum(acc_l ? log(fabs(R_l)) : 0.0);     // fixed (butterfly) order
        const unsigned neg = __ballot_sync(0xffffffffu, acc_l && R_l < 0.0);
        if (lane == 0) {
            if (a.cur) { a.cur[w] = iel0 + nproc; a.ev[w] = iel0 + nb; }
            a.win_count[w] = p;
            p_s = p;
            if (p) {
                a.logdet[w] += logdet_add;
                if (__popc(neg) & 1) a.sign[w] = -a.sign[w];
                a.naccept[w] += p;
            }
        }
        if (lane < p) {
            a.win_iel[(size_t)w * K + lane] = iel0 + mine;
            a.win_slot[(size_t)w * K + lane] = ring ? (iel0 + mine) % ring : mine;
            rowoff_s[lane] = (long long)mine * ld;
        }
    }
    __syncthreads();

    // ---- phase 4: R'[l] = sum_l' S^-1[l'][l] B0[k_l'] for the flush (pad columns of B are zero)
    const int p = p_s;
    if (p) rprime_warp<PMAX, TB>(sinv_s, GS, p, b0, rowoff_s, a.win_rows + (size_t)w * K * ld, ld, warp, kWinThreads / 32, lane);
}

int delayed_sweep_window(qmc_det *d, double *pos, const double *delta, const double *unif, int iel0, int nb,
                         double *ratios_out, unsigned char *accept_out, const unsigned char *forced,
                         int fixed_node, double *force_out, int record_mid, const WindowJastrow &jas, cudaStream_t s)
{
    if (d->host_pending) {        // rows pending from standalone qmc_det_accept_update calls
        int rc = delayed_flush_reset_host(d, s);
        if (rc) return rc;
    }
    WindowArgs a{};
    a.B = d->b32 ? (const void *)d->Bf : (const void *)d->B;
    a.nw = d->nw; a.nel = d->nel; a.ld = d->ld; a.np = d->np; a.K = d->delay;
    a.iel0 = iel0; a.nb = nb;
    a.vgl = d->vgl;
    a.unif = unif; a.forced = forced; a.ratios_out = ratios_out; a.accept_out = accept_out;
    a.fixed_node = fixed_node; a.force_out = force_out;
    a.pos = pos; a.delta = delta;
    a.logdet = d->logdet; a.sign = d->sign; a.naccept = d->naccept;
    a.win_count = d->win_count; a.win_iel = d->win_iel; a.win_slot = d->win_slot;
    a.win_rows = d->win_rows;
    a.jas = jas;
    a.pmax = d->delay;
    if (d->accept_windows) { a.cur = d->cur; a.ev = d->cur + d->nw; a.kend = d->win_kend; a.ring = d->vgl_ring; }
    const int kwin = d->accept_windows ? d->spo_batch : a.K;     // steps per window: what the G matrix must hold
    prof_start(d, kProfDelayedRatio, s);
#define QMC_WIN_LAUNCH(TB, KM, F, J) delayed_window_kernel<TB, KM, F, J><<<d->nw, kWinThreads, 0, s>>>(a)
#define QMC_WIN_LAUNCH_P(TB, KM, F, J, PM) delayed_window_kernel<TB, KM, F, J, PM><<<d->nw, kWinThreads, 0, s>>>(a)
#define QMC_WIN_RANK(TB, F, J)                               \
    do {                                                     \
        if (kwin <= 8) QMC_WIN_LAUNCH(TB, 8, F, J);          \
        else if (kwin <= 16) QMC_WIN_LAUNCH(TB, 16, F, J);   \
        else if (kwin <= 24 && a.pmax <= 16) QMC_WIN_LAUNCH_P(TB, 24, F, J, 16); \
        else if (kwin <= 24) QMC_WIN_LAUNCH(TB, 24, F, J);   \
        else QMC_WIN_LAUNCH(TB, 32, F, J);                   \
    } while (0)
#define QMC_WIN_JAS(TB, F)                                   \
    do {                                                     \
        if (jas.base) QMC_WIN_RANK(TB, F, true);            \
        else QMC_WIN_RANK(TB, F, false);                     \
    } while (0)
    if (d->b32) { if (force_out) QMC_WIN_JAS(float, true); else QMC_WIN_JAS(float, false); }
    else { if (force_out) QMC_WIN_JAS(double, true); else QMC_WIN_JAS(double, false); }
#undef QMC_WIN_JAS
#undef QMC_WIN_RANK
#undef QMC_WIN_LAUNCH_P
#undef QMC_WIN_LAUNCH
    prof_stop(d, s);
    QMC_LAUNCHED();
    // positions are final for this window: the next window's SPO-VGL may start (second stream, sweep.cu)
    if (record_mid) QMC_CUDA(cudaEventRecord(d->ev_main, s));
    // the flush takes the vectors of the accepted steps straight from the SPO-VGL scratch
    d->host_pending = nb;
    d->win_rows_raw = 0;
    d->win_vec = d->vgl;
    d->win_vec_wstride = (size_t)5 * d->np;
    d->win_vec_sstride = (size_t)d->nw * 5 * d->np;
    return delayed_flush_reset_host(d, s);
}

}  // namespace qmc
