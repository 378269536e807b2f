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
// A window is K consecutive electron steps of the lockstep sweep (R:A14), so the host schedules
// the flushes and no device -> host traffic is needed.
#include "delayed_device.cuh"
#include "spo_device.cuh"
#include "update_device.cuh"

namespace qmc {

void spo_launch_shape(int np, int *threads, int *tiles);

constexpr int kStepThreads = 256;

struct DelayedStepArgs {
    const double *B;              // [nw][nel][ld]  (B0 during a window)
    int nel, ld, np, iel, K;
    const float *phi;             // [nw][ldphi]
    size_t ldphi;
    // window state
    int *win_count;               // [nw]
    int *win_iel;                 // [nw][K]
    float *win_phi;               // [nw][K][np]
    double *win_rows;             // [nw][K][ld]
    double *win_sinv;             // [nw][K][K]
    // mode: decide here (sweep) or ratio only / accept only (standalone API)
    int mode;                     // 0 = sweep step (ratio + decide + append), 1 = ratio only, 2 = append only
    double *ratio_io;             // [nw]  mode 1: out; mode 2: in
    const unsigned char *accept_in;   // [nw] mode 2
    const double *unif;           // [nw]  mode 0
    const unsigned char *forced;  // [nw] or NULL, mode 0
    double *ratios_out;           // [nw] or NULL, mode 0
    unsigned char *accept_out;    // [nw] or NULL, mode 0
    double *pos;                  // [nw][nel][3], mode 0
    const double *delta;          // [nw][3], mode 0
    double *logdet;
    int *sign;
    long long *naccept;
};

// One block per walker.  Each thread owns column quads j = 4*tid (+ 4*blockDim per pass): it
// accumulates the 2p+1 partial dots d, x_m, c_l over its columns; the block reduces them in a
// fixed order; warp 0 finishes the ratio, takes the Metropolis decision and, on accept, grows the
// window (row copy, orbital vector copy, bordered S^-1).
template <int KMAX>
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
    const double *b0k = a.B + ((size_t)w * a.nel + a.iel) * ld;
    const float *phi = a.phi + (size_t)w * a.ldphi;
    const double *rows = a.win_rows + (size_t)w * K * ld;
    const float *vwin = a.win_phi + (size_t)w * K * np;

    double acc[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) acc[i] = 0.0;
    {
        for (int j = 4 * tid; j < np; j += 4 * kStepThreads) {
            const float4 f = *reinterpret_cast<const float4 *>(phi + j);
            const double2 ba = *reinterpret_cast<const double2 *>(b0k + j);
            const double2 bb = *reinterpret_cast<const double2 *>(b0k + j + 2);
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
        if (a.mode == 2) {
            acc_w = a.accept_in[w] != 0;      // the caller's decision; R equals the ratio it was given
        } else if (a.mode == 0) {
            acc_w = a.forced ? (a.forced[w] != 0) : metropolis(R, a.unif[w]);
            if (a.ratios_out) a.ratios_out[w] = R;
            if (a.accept_out) a.accept_out[w] = acc_w ? 1 : 0;
        } else {
            a.ratio_io[w] = R;
        }
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
        if (a.mode == 0) {
            double *r = a.pos + ((size_t)w * a.nel + a.iel) * 3;
            r[0] += a.delta[3 * (size_t)w + 0];
            r[1] += a.delta[3 * (size_t)w + 1];
            r[2] += a.delta[3 * (size_t)w + 2];
        }
        a.win_iel[(size_t)w * K + p] = a.iel;
        a.win_count[w] = p + 1;
    }
    // append the orbital vector and the row B0[k]
    float *vdst = a.win_phi + ((size_t)w * K + p) * np;
    double *rdst = a.win_rows + ((size_t)w * K + p) * ld;
    for (int j = 4 * tid; j < np; j += 4 * kStepThreads)
        *reinterpret_cast<float4 *>(vdst + j) = *reinterpret_cast<const float4 *>(phi + j);
    for (int j = 2 * tid; j < ld; j += 2 * kStepThreads)
        *reinterpret_cast<double2 *>(rdst + j) = *reinterpret_cast<const double2 *>(b0k + j);
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

// ---------------------------------------------------------------------------------------------
// flush

// Reduce NV (power of two <= 32) per-lane partials across the warp with NV-1 + log2(32/NV)
// shuffle-adds; afterwards lane L holds the total of value L / (32 / NV).  Fixed order.
template <int NV>
__device__ __forceinline__ double warp_multi_reduce(double (&v)[NV])
{
    const int lane = threadIdx.x & 31;
    int n = NV;
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        if (n > 1) {
            n >>= 1;
            const bool upper = (lane & off) != 0;
#pragma unroll
            for (int i = 0; i < NV / 2; ++i) {
                if (i < n) {
                    const double send = upper ? v[i] : v[i + n];
                    const double keep = upper ? v[i + n] : v[i];
                    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
                }
            }
        } else {
            v[0] += __shfl_xor_sync(0xffffffffu, v[0], off);
        }
    }
    return v[0];
}

struct FlushArgs {
    double *B;                    // [nw][nel][ld]
    int nel, ld, np, K;
    const int *win_count;
    const int *win_iel;
    const float *win_phi;
    const double *win_rows;
    const double *win_sinv;
};

constexpr int kFlushThreads = 256;
constexpr int kFlushRowsPerCta = 64;

// Single pass over B.  The window's orbital vectors (fp32) and saved rows (fp64) live in shared
// memory for the whole CTA; a warp keeps RPW rows of B in registers, forms their p dots with the
// vectors (multi-value butterfly reduction), multiplies by S^-1, and subtracts the p saved rows.
template <int VPT, int KPAD, int RPW>
__global__ void __launch_bounds__(kFlushThreads, 1) delayed_flush_kernel(FlushArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_flush[];
    const int w = blockIdx.y;
    const int p = a.win_count[w];
    if (p == 0) return;
    const int ld = a.ld, K = a.K, np = a.np;
    double *rows_s = reinterpret_cast<double *>(smem_flush);                    // [K][ld]
    float *v_s = reinterpret_cast<float *>(rows_s + (size_t)K * ld);            // [K][ld]
    double *sinv_s = reinterpret_cast<double *>(v_s + (size_t)K * ld);          // [KPAD][KPAD]
    int *kl_s = reinterpret_cast<int *>(sinv_s + KPAD * KPAD);                  // [KPAD]
    const double *rows_g = a.win_rows + (size_t)w * K * ld;
    const float *v_g = a.win_phi + (size_t)w * K * np;
    for (int e = threadIdx.x; e < p * (ld / 2); e += kFlushThreads) {
        const int l = e / (ld / 2), c = e % (ld / 2);
        reinterpret_cast<double2 *>(rows_s + (size_t)l * ld)[c] =
            reinterpret_cast<const double2 *>(rows_g + (size_t)l * ld)[c];
        float2 f = make_float2(0.f, 0.f);
        if (2 * c < np) f = reinterpret_cast<const float2 *>(v_g + (size_t)l * np)[c];
        reinterpret_cast<float2 *>(v_s + (size_t)l * ld)[c] = f;
    }
    for (int e = threadIdx.x; e < KPAD * KPAD; e += kFlushThreads) {
        const int i = e / KPAD, j = e % KPAD;
        sinv_s[e] = (i < p && j < p) ? a.win_sinv[(size_t)w * K * K + i * K + j] : 0.0;
    }
    if (threadIdx.x < KPAD) kl_s[threadIdx.x] = threadIdx.x < p ? a.win_iel[(size_t)w * K + threadIdx.x] : -1;
    __syncthreads();

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    constexpr int NV = KPAD * RPW;                 // partials per lane, <= 32
    constexpr int LPV = 32 / NV;                   // lanes per value after the reduction
    const int my_val = lane / LPV;                 // value index this lane ends up holding
    const int my_row = my_val / KPAD, my_l = my_val % KPAD;
    const int m_begin = blockIdx.x * kFlushRowsPerCta, m_end = min(a.nel, m_begin + kFlushRowsPerCta);
    for (int m0 = m_begin + wid * RPW; m0 < m_end; m0 += (kFlushThreads / 32) * RPW) {
        double2 r[RPW][VPT];
#pragma unroll
        for (int q = 0; q < RPW; ++q) {
            const int m = min(m0 + q, a.nel - 1);
            const double2 *row = reinterpret_cast<const double2 *>(a.B + ((size_t)w * a.nel + m) * ld);
#pragma unroll
            for (int i = 0; i < VPT; ++i) r[q][i] = row[lane + 32 * i];
        }
        double part[NV];
#pragma unroll
        for (int i = 0; i < NV; ++i) part[i] = 0.0;
#pragma unroll
        for (int l = 0; l < KPAD; ++l) {
            if (l < p) {
                const float2 *vl = reinterpret_cast<const float2 *>(v_s + (size_t)l * ld);
#pragma unroll
                for (int i = 0; i < VPT; ++i) {
                    const float2 f = vl[lane + 32 * i];
                    const double fx = f.x, fy = f.y;
#pragma unroll
                    for (int q = 0; q < RPW; ++q)
                        part[q * KPAD + l] = fma(r[q][i].x, fx, fma(r[q][i].y, fy, part[q * KPAD + l]));
                }
            }
        }
        // lane holds q_{my_l}(row my_row)
        double qv = warp_multi_reduce<NV>(part);
        if (my_l < p && kl_s[my_l] == m0 + my_row) qv -= 1.0;
        // t_l = sum_l' S^-1[l][l'] q_l'   (lane computes the t of its own (row, l))
        double t = 0.0;
#pragma unroll
        for (int l2 = 0; l2 < KPAD; ++l2) {
            const double ql = __shfl_sync(0xffffffffu, qv, (my_row * KPAD + l2) * LPV);
            t = fma(sinv_s[my_l * KPAD + l2], ql, t);
        }
#pragma unroll
        for (int l = 0; l < KPAD; ++l) {
            if (l < p) {
                double tl[RPW];
#pragma unroll
                for (int q = 0; q < RPW; ++q) tl[q] = __shfl_sync(0xffffffffu, t, (q * KPAD + l) * LPV);
                const double2 *rl = reinterpret_cast<const double2 *>(rows_s + (size_t)l * ld);
#pragma unroll
                for (int i = 0; i < VPT; ++i) {
                    const double2 k2 = rl[lane + 32 * i];
#pragma unroll
                    for (int q = 0; q < RPW; ++q) {
                        r[q][i].x = fma(-tl[q], k2.x, r[q][i].x);
                        r[q][i].y = fma(-tl[q], k2.y, r[q][i].y);
                    }
                }
            }
        }
#pragma unroll
        for (int q = 0; q < RPW; ++q) {
            if (m0 + q < m_end) {
                double2 *row = reinterpret_cast<double2 *>(a.B + ((size_t)w * a.nel + m0 + q) * ld);
#pragma unroll
                for (int i = 0; i < VPT; ++i) row[lane + 32 * i] = r[q][i];
            }
        }
    }
}

__global__ void reset_window_kernel(int nw, int *win_count)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < nw) win_count[w] = 0;
}

static size_t flush_smem_bytes(int K, int kpad, int ld)
{
    return (size_t)K * ld * (sizeof(double) + sizeof(float)) + (size_t)kpad * kpad * sizeof(double) +
           (size_t)kpad * sizeof(int);
}

static int kpad_of(int K) { int k = 2; while (k < K) k <<= 1; return k; }

// Largest delay rank whose window fits the flush kernel's shared memory for this ld.
int delayed_max_rank(int ld)
{
    int best = 0;
    for (int K = 2; K <= QMC_MAX_DELAY; ++K)
        if (flush_smem_bytes(K, kpad_of(K), ld) <= 227 * 1024) best = K;
    return best;
}

template <int VPT, int KPAD, int RPW>
static cudaError_t launch_flush_t(const FlushArgs &a, int nw, size_t smem, cudaStream_t s)
{
    auto kern = delayed_flush_kernel<VPT, KPAD, RPW>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((a.nel + kFlushRowsPerCta - 1) / kFlushRowsPerCta, nw);
    kern<<<grid, kFlushThreads, smem, s>>>(a);
    return cudaGetLastError();
}

template <int VPT>
static cudaError_t launch_flush_v(const FlushArgs &a, int nw, cudaStream_t s)
{
    const int kpad = kpad_of(a.K);
    const size_t smem = flush_smem_bytes(a.K, kpad, a.ld);
    constexpr bool two = VPT <= 16;
    switch (kpad) {
    case 2: return launch_flush_t<VPT, 2, two ? 2 : 1>(a, nw, smem, s);
    case 4: return launch_flush_t<VPT, 4, two ? 2 : 1>(a, nw, smem, s);
    case 8: return launch_flush_t<VPT, 8, two ? 2 : 1>(a, nw, smem, s);
    case 16: return launch_flush_t<VPT, 16, two ? 2 : 1>(a, nw, smem, s);
    case 32: return launch_flush_t<VPT, 32, 1>(a, nw, smem, s);
    }
    return cudaErrorInvalidValue;
}

int delayed_flush(qmc_det *d, cudaStream_t s)
{
    if (!d->delay || d->host_pending == 0) return QMC_OK;
    FlushArgs a{};
    a.B = d->B; a.nel = d->nel; a.ld = d->ld; a.np = d->np; a.K = d->delay;
    a.win_count = d->win_count; a.win_iel = d->win_iel; a.win_phi = d->win_phi;
    a.win_rows = d->win_rows; a.win_sinv = d->win_sinv;
    cudaError_t e;
    prof_start(d, kProfDelayedFlush, s);
    switch (d->ld / 64) {
#define QMC_FL_CASE(V) case V: e = launch_flush_v<V>(a, d->nw, s); break;
        QMC_FL_CASE(1) QMC_FL_CASE(2) QMC_FL_CASE(3) QMC_FL_CASE(4) QMC_FL_CASE(6)
        QMC_FL_CASE(8) QMC_FL_CASE(12) QMC_FL_CASE(16) QMC_FL_CASE(24) QMC_FL_CASE(32)
#undef QMC_FL_CASE
    default: e = cudaErrorInvalidValue;
    }
    prof_stop(d, s);
    count_launch();
    QMC_CUDA(e);
    reset_window_kernel<<<(d->nw + 127) / 128, 128, 0, s>>>(d->nw, d->win_count);
    QMC_LAUNCHED();
    d->host_pending = 0;
    return QMC_OK;
}

static cudaError_t launch_step(const DelayedStepArgs &a, int nw, cudaStream_t s)
{
    if (a.K <= 8) delayed_step_kernel<8><<<nw, kStepThreads, 0, s>>>(a);
    else if (a.K <= 16) delayed_step_kernel<16><<<nw, kStepThreads, 0, s>>>(a);
    else delayed_step_kernel<32><<<nw, kStepThreads, 0, s>>>(a);
    count_launch();
    return cudaGetLastError();
}

static void fill_common(DelayedStepArgs &a, qmc_det *d, int iel, const float *phi, size_t ldphi)
{
    a.B = d->B; a.nel = d->nel; a.ld = d->ld; a.np = d->np; a.iel = iel; a.K = d->delay;
    a.phi = phi; a.ldphi = ldphi;
    a.win_count = d->win_count; a.win_iel = d->win_iel; a.win_phi = d->win_phi;
    a.win_rows = d->win_rows; a.win_sinv = d->win_sinv;
    a.logdet = d->logdet; a.sign = d->sign; a.naccept = d->naccept;
}

int delayed_ratio(qmc_det *d, int iel, const float *phi, int ldo, double *ratio, cudaStream_t s)
{
    QMC_REQUIRE(ldo >= d->np, "qmc_det_ratio (delayed): ldo=%d must be >= the table pitch %d", ldo, d->np);
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
    cudaError_t e = launch_step(a, d->nw, s);
    prof_stop(d, s);
    QMC_CUDA(e);
    return QMC_OK;
}

int delayed_accept(qmc_det *d, int iel, const float *phi, int ldo, const double *ratio,
                   const unsigned char *accept, cudaStream_t s)
{
    QMC_REQUIRE(ldo >= d->np, "qmc_det_accept_update (delayed): ldo=%d must be >= the table pitch %d", ldo, d->np);
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
    cudaError_t e = launch_step(a, d->nw, s);
    prof_stop(d, s);
    QMC_CUDA(e);
    d->host_pending += 1;
    d->win_host_iel[iel] = 1;
    return QMC_OK;
}

int delayed_flush_reset_host(qmc_det *d, cudaStream_t s)
{
    int rc = delayed_flush(d, s);
    if (rc) return rc;
    if (d->win_host_iel) memset(d->win_host_iel, 0, (size_t)d->nel);
    return QMC_OK;
}

int delayed_sweep_step(qmc_det *d, const qmc_spline *sp, double *pos, const double *delta, const double *unif,
                       int iel, double *ratios_out, unsigned char *accept_out, const unsigned char *forced,
                       float *phi_record, int nrecord, cudaStream_t s)
{
    if (d->host_pending >= d->delay || (d->host_pending && d->win_host_iel[iel])) {
        int rc = delayed_flush_reset_host(d, s);
        if (rc) return rc;
    }
    // K1: SPO-VGL at the proposed positions (into the walker scratch), K2: ratio / decide / append
    int rc = spo_proposal_vgl(d, sp, pos, delta, iel, phi_record, nrecord, s);
    if (rc) return rc;
    DelayedStepArgs a{};
    fill_common(a, d, iel, d->vgl, (size_t)5 * d->np);
    a.mode = 0;
    a.unif = unif; a.forced = forced; a.ratios_out = ratios_out; a.accept_out = accept_out;
    a.pos = pos; a.delta = delta;
    prof_start(d, kProfDelayedRatio, s);
    cudaError_t e = launch_step(a, d->nw, s);
    prof_stop(d, s);
    QMC_CUDA(e);
    d->host_pending += 1;
    d->win_host_iel[iel] = 1;
    return QMC_OK;
}

}  // namespace qmc
