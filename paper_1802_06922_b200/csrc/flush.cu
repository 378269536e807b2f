// Flush of the delayed (rank-k) update as two dense fp64 contractions on the tensor cores
// ("a delayed update algorithm that enables increased use of matrix-matrix
// multiplication [44]", L299; formulas: DESIGN.md section 3, R:O7):
//
//     Q[m][l] = B0[m] . v_l - [k_l == m]          (N x N)(N x p)     step 1
//     T       = Q S^-T                             (N x p)(p x p)
//     B[m]    = B0[m] - sum_l T[m][l] * B0[k_l]    (N x p)(p x N)     step 2
//
// in ONE pass over B (16 N ld bytes per walker): a warp keeps an 8-row x (8 TW)-column block of B
// in registers.  With the contraction index of step 1 permuted so that one lane's `double2` of a
// row serves two consecutive k-steps, the registers a lane loads (row g, columns 2t, 2t+1 of every
// 8-column tile) are at once the A fragments of step 1 and the C fragments of step 2 of
// mma.sync.m8n8k4.f64 (SASS: DMMA.8x8x4), and T's C fragments are step 2's A fragments when its
// contraction index is permuted the same way: no shuffles, no transposes.
//
// The walker's window (p saved rows in fp64, p orbital vectors in fp32, S^-1) is staged once per
// CTA into shared memory with TMA bulk copies (cp.async.bulk + mbarrier) and shared by NG warp
// groups that stream different row blocks out of phase, so one group's DMMA work overlaps the
// other group's HBM loads and stores.
#include "delayed_device.cuh"

namespace qmc {

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
    } while (!ok);
}
// TMA 1-D bulk copy global -> shared, completion counted on `bar` (bytes % 16 == 0, 16-B aligned).
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void group_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
struct FlushArgs {
    double *B;                    // [nw][nel][ld]
    int nel, ld, np, K;
    int rows_per_cta;             // multiple of 8 * NG
    const int *win_count;
    const int *win_iel;
    const float *win_phi;
    const double *win_rows;
    const double *win_sinv;
};

// Shared-memory geometry (strides chosen so every fragment load is bank-conflict free):
//   rows_s  double [KPAD][LD + 2]   B-fragment of step 2: lane (g,t) reads row 8nt+2t+h, column n0+g
//   v_s     float  [KPAD][LD + 8]   B-fragment of step 1: lane (g,t) reads row 8nt+g, columns n0+2t,+1
//   sinv_s  double [KPAD][KPAD + 4]
//   part_s  double [2][NG][NWC][8][KPAD + 4]   partial Q of each column warp, by block parity
//   kl_s    int [KPAD],  mbar
template <int KPAD, int LD, int NWC, int NG>
struct FlushSmem {
    static constexpr int RS = LD + 2, VS = LD + 8, SS = KPAD + 4, PS = KPAD + 4;
    static constexpr size_t rows_off = 0;
    static constexpr size_t v_off = rows_off + (size_t)KPAD * RS * sizeof(double);
    static constexpr size_t sinv_off = v_off + (size_t)KPAD * VS * sizeof(float);
    static constexpr size_t part_off = sinv_off + (size_t)KPAD * SS * sizeof(double);
    static constexpr size_t part_bytes = (size_t)NG * NWC * 8 * PS * sizeof(double);
    // two partial buffers (by block parity) save a barrier per block; one when shared memory is short
    static constexpr int PB = (part_off + 2 * part_bytes + KPAD * sizeof(int) + 16 <= 227 * 1024) ? 2 : 1;
    static constexpr size_t kl_off = part_off + PB * part_bytes;
    static constexpr size_t mbar_off = kl_off + (size_t)KPAD * sizeof(int);
    static constexpr size_t bytes = mbar_off + 16;
};

constexpr size_t kSmemMax = 227 * 1024;

template <int KPAD, int NWC, int TW, int NG, bool PF>
__global__ void __launch_bounds__(32 * NWC * NG, 1) flush_dmma_kernel(FlushArgs a)
{
    constexpr int LD = NWC * TW * 8;
    constexpr int NT = KPAD / 8;
    using L = FlushSmem<KPAD, LD, NWC, NG>;
    constexpr int RS = L::RS, VS = L::VS, SS = L::SS, PS = L::PS;
    constexpr int NTHREADS = 32 * NWC * NG;
    extern __shared__ __align__(128) unsigned char smem_flush[];
    double *rows_s = reinterpret_cast<double *>(smem_flush + L::rows_off);
    float *v_s = reinterpret_cast<float *>(smem_flush + L::v_off);
    double *sinv_s = reinterpret_cast<double *>(smem_flush + L::sinv_off);
    double *part_s = reinterpret_cast<double *>(smem_flush + L::part_off);
    int *kl_s = reinterpret_cast<int *>(smem_flush + L::kl_off);
    uint64_t *mbar = reinterpret_cast<uint64_t *>(smem_flush + L::mbar_off);

    const int w = blockIdx.y;
    const int p = a.win_count[w];
    if (p == 0) return;
    const int p8 = (p + 7) & ~7;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int grp = warp / NWC, wc = warp % NWC;
    const int K = a.K, np = a.np, nel = a.nel;

    // ---- stage the window: zero what the bulk copies do not write, then TMA the rows in
    if (tid == 0) mbar_init(mbar, 1);
    for (int e = tid; e < p * (LD - np); e += NTHREADS) {          // pad columns of the vectors
        const int l = e / (LD - np), c = np + e % (LD - np);
        v_s[l * VS + c] = 0.f;
    }
    for (int e = tid; e < (p8 - p) * LD; e += NTHREADS) {          // rows p..p8-1 of the last tile
        const int l = p + e / LD, c = e % LD;
        v_s[l * VS + c] = 0.f;
        rows_s[l * RS + c] = 0.0;
    }
    for (int e = tid; e < KPAD * KPAD; e += NTHREADS) {
        const int i = e / KPAD, j = e % KPAD;
        sinv_s[i * SS + j] = (i < p && j < p) ? a.win_sinv[(size_t)w * K * K + i * K + j] : 0.0;
    }
    if (tid < KPAD) kl_s[tid] = tid < p ? a.win_iel[(size_t)w * K + tid] : -1;
    __syncthreads();
    if (warp == 0) {
        if (lane == 0) mbar_arrive_expect_tx(mbar, (uint32_t)p * (uint32_t)(LD * sizeof(double) + np * sizeof(float)));
        __syncwarp();
        const double *rows_g = a.win_rows + (size_t)w * K * LD;
        const float *v_g = a.win_phi + (size_t)w * K * np;
        for (int l = lane; l < p; l += 32) {
            bulk_g2s(rows_s + l * RS, rows_g + (size_t)l * LD, LD * sizeof(double), mbar);
            bulk_g2s(v_s + l * VS, v_g + (size_t)l * np, np * sizeof(float), mbar);
        }
    }

    // ---- stream row blocks: group `grp` takes blocks grp, grp + NG, ... of this CTA's rows.
    // With PF the next block's rows are requested before the current block is contracted, so the
    // HBM stream (loads of block i+1, stores of block i-1) runs under the DMMA work of block i.
    const int m_begin = blockIdx.x * a.rows_per_cta;
    const int m_end = min(nel, m_begin + a.rows_per_cta);
    const int col0 = 8 * TW * wc;
    double *const walker_B = a.B + (size_t)w * nel * LD + col0 + 2 * t;
    bool staged = false;
    int m0 = m_begin + 8 * grp;
    double2 r[TW], rn[PF ? TW : 1];
    if (m0 < m_end) {
        const double *src = walker_B + (size_t)min(m0 + g, nel - 1) * LD;
#pragma unroll
        for (int i = 0; i < TW; ++i) r[i] = *reinterpret_cast<const double2 *>(src + 8 * i);
    }
    for (int it = 0; m0 < m_end; m0 += 8 * NG, ++it) {
        const int m = m0 + g;
        const int m0n = m0 + 8 * NG;
        if (PF && m0n < m_end) {
            const double *src = walker_B + (size_t)min(m0n + g, nel - 1) * LD;
#pragma unroll
            for (int i = 0; i < TW; ++i) rn[PF ? i : 0] = *reinterpret_cast<const double2 *>(src + 8 * i);
        }
        if (!staged) {
            mbar_wait(mbar, 0);
            staged = true;
        }
        // step 1: partial Q over this warp's columns
        double cq[NT][2];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) cq[nt][0] = cq[nt][1] = 0.0;
#pragma unroll
        for (int i = 0; i < TW; ++i) {
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
                if (8 * nt < p) {
                    const float2 f = *reinterpret_cast<const float2 *>(v_s + (8 * nt + g) * VS + col0 + 8 * i + 2 * t);
                    dmma884(cq[nt][0], cq[nt][1], r[i].x, (double)f.x);
                    dmma884(cq[nt][0], cq[nt][1], r[i].y, (double)f.y);
                }
            }
        }
        // partials are double-buffered by block parity: one barrier per block is enough
        double *pbuf = part_s + (size_t)((L::PB == 2 ? (it & 1) : 0) * NG + grp) * NWC * 8 * PS;
        double *ps = pbuf + ((size_t)wc * 8 + g) * PS;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
            if (8 * nt < p) *reinterpret_cast<double2 *>(ps + 8 * nt + 2 * t) = make_double2(cq[nt][0], cq[nt][1]);
        group_sync(1 + grp, 32 * NWC);
        // Q as A fragments: lane (g,t), k-step k' holds Q[m0+g][4k'+t], summed over the column warps
        double qa[KPAD / 4];
#pragma unroll
        for (int kq = 0; kq < KPAD / 4; ++kq) {
            double s = 0.0;
            if (4 * kq < p8) {
                const double *pp = pbuf + (size_t)g * PS + 4 * kq + t;
#pragma unroll
                for (int c = 0; c < NWC; ++c) s += pp[(size_t)c * 8 * PS];
                if (kl_s[4 * kq + t] == m) s -= 1.0;
            }
            qa[kq] = s;
        }
        if (L::PB == 1) group_sync(1 + grp, 32 * NWC);
        // T = Q S^-T (C fragments), negated
        double tq[NT][2];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            tq[nt][0] = tq[nt][1] = 0.0;
            if (8 * nt < p) {
#pragma unroll
                for (int kq = 0; kq < KPAD / 4; ++kq)
                    if (4 * kq < p8) dmma884(tq[nt][0], tq[nt][1], qa[kq], sinv_s[(8 * nt + g) * SS + 4 * kq + t]);
            }
        }
        // step 2: B block += (-T) Rows; contraction index l = 8nt + 2t + h
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            if (8 * nt < p) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const double af = -tq[nt][h];
                    const double *rp = rows_s + (8 * nt + 2 * t + h) * RS + col0 + g;
#pragma unroll
                    for (int i = 0; i < TW; ++i) dmma884(r[i].x, r[i].y, af, rp[8 * i]);
                }
            }
        }
        if (m < nel) {
            double *dst = walker_B + (size_t)m * LD;
#pragma unroll
            for (int i = 0; i < TW; ++i) *reinterpret_cast<double2 *>(dst + 8 * i) = r[i];
        }
        if (PF) {
#pragma unroll
            for (int i = 0; i < TW; ++i) r[i] = rn[PF ? i : 0];
        } else if (m0n < m_end) {
            const double *src = walker_B + (size_t)min(m0n + g, nel - 1) * LD;
#pragma unroll
            for (int i = 0; i < TW; ++i) r[i] = *reinterpret_cast<const double2 *>(src + 8 * i);
        }
    }
    if (!staged) mbar_wait(mbar, 0);            // never leave with bulk copies in flight
}

__global__ void reset_window_kernel(int nw, int *win_count)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < nw) win_count[w] = 0;
}

// Launch shape for ld = 64 v: NWC column warps x TW 8-column tiles per warp, NG row groups per
// CTA, PF = prefetch the next row block (needs 2 x 4 TW data registers per thread).
struct FlushShape { int nwc, tw, ng; };
#define QMC_FLUSH_SHAPES(X) \
    X(1, 1, 8, 4, true) X(2, 2, 8, 4, true) X(3, 3, 8, 4, true) X(4, 4, 8, 4, true) X(6, 6, 8, 2, true) \
    X(8, 8, 8, 2, true) X(12, 6, 16, 2, false) X(16, 8, 16, 2, false) X(24, 12, 16, 1, false) X(32, 16, 16, 1, false)

static FlushShape flush_shape(int v)
{
    switch (v) {
#define X(V, NWC, TW, NG, PF) case V: return {NWC, TW, NG};
        QMC_FLUSH_SHAPES(X)
#undef X
    }
    return {0, 0, 0};
}

static int kpad_of(int K) { return (K + 7) / 8 * 8; }

static size_t flush_smem_bytes(int kpad, int ld)
{
    const FlushShape s = flush_shape(ld / 64);
    return (size_t)kpad * (ld + 2) * 8 + (size_t)kpad * (ld + 8) * 4 + (size_t)kpad * (kpad + 4) * 8 +
           (size_t)s.ng * s.nwc * 8 * (kpad + 4) * 8 + (size_t)kpad * 4 + 16;
}

// Largest delay rank whose window fits the flush kernel's shared memory for this ld.
int delayed_max_rank(int ld)
{
    int best = 0;
    for (int K = 2; K <= QMC_MAX_DELAY; ++K)
        if (flush_smem_bytes(kpad_of(K), ld) <= kSmemMax) best = K;
    return best;
}

template <int KPAD, int NWC, int TW, int NG, bool PF>
static cudaError_t launch_flush_t(const FlushArgs &a, int nw, cudaStream_t s)
{
    using L = FlushSmem<KPAD, NWC * TW * 8, NWC, NG>;
    if constexpr (L::bytes > kSmemMax) {
        return cudaErrorInvalidValue;
    } else {
        auto kern = flush_dmma_kernel<KPAD, NWC, TW, NG, PF>;
        static bool configured = false;
        if (!configured) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::bytes);
            if (e != cudaSuccess) return e;
            configured = true;
        }
        dim3 grid((a.nel + a.rows_per_cta - 1) / a.rows_per_cta, nw);
        kern<<<grid, 32 * NWC * NG, L::bytes, s>>>(a);
        return cudaGetLastError();
    }
}

template <int NWC, int TW, int NG, bool PF>
static cudaError_t launch_flush_k(const FlushArgs &a, int nw, cudaStream_t s)
{
    switch (kpad_of(a.K)) {
    case 8: return launch_flush_t<8, NWC, TW, NG, PF>(a, nw, s);
    case 16: return launch_flush_t<16, NWC, TW, NG, PF>(a, nw, s);
    case 24: return launch_flush_t<24, NWC, TW, NG, PF>(a, nw, s);
    case 32: return launch_flush_t<32, NWC, TW, NG, PF>(a, nw, s);
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
    const FlushShape sh = flush_shape(d->ld / 64);
    // rows per CTA: the window is staged once per CTA, so prefer long CTAs when the grid stays large
    a.rows_per_cta = ((long long)d->nw * d->nel >= 128LL * 148 * 8) ? 128 : 64;
    if (a.rows_per_cta % (8 * sh.ng)) a.rows_per_cta = 8 * sh.ng * ((a.rows_per_cta + 8 * sh.ng - 1) / (8 * sh.ng));
    cudaError_t e;
    prof_start(d, kProfDelayedFlush, s);
    switch (d->ld / 64) {
#define X(V, NWC, TW, NG, PF) case V: e = launch_flush_k<NWC, TW, NG, PF>(a, d->nw, s); break;
        QMC_FLUSH_SHAPES(X)
#undef X
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

}  // namespace qmc
