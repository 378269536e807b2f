// Flush of the delayed (rank-k) update as two dense fp64 contractions on the tensor cores
// ("a delayed update algorithm that enables increased use of matrix-matrix
// multiplication [44]", L299; formulas: DESIGN.md section 3, R:O7):
//
//     Q[m][l] = B0[m] . v_l - [k_l == m]          (N x N)(N x p)     step 1
//     B[m]    = B0[m] - sum_l Q[m][l] * R'[l]      (N x p)(p x N)     step 2,  R' = S^-T Rows
//
// in ONE pass over B (16 N ld bytes per walker): a warp keeps an 8-row x (8 TW)-column block of B
// in registers.  With the contraction index of step 1 permuted so that one lane's `double2` of a
// row serves two consecutive k-steps, the registers a lane loads (row g, columns 2t, 2t+1 of every
// 8-column tile) are at once the A fragments of step 1 and the C fragments of step 2 of
// mma.sync.m8n8k4.f64 (SASS: DMMA.8x8x4); Q, summed over the column slices, is read back from
// shared memory directly in A-fragment layout for step 2: no shuffles, no transposes.
//
// The walker's window (p rows of R' in fp64, p orbital vectors in fp32) is staged once per CTA into
// shared memory with TMA bulk copies (cp.async.bulk + mbarrier).  For large N the columns of a row
// block are split over a thread-block CLUSTER (each CTA stages only its column slice of the window,
// so two or three CTAs fit an SM and one CTA's HBM stream runs under another's DMMA work); the
// partial Q of the slices are exchanged through distributed shared memory once per row block.
#include <stdlib.h>
#include "delayed_device.cuh"
#include "async_device.cuh"
#include "dmma.cuh"

namespace qmc {

struct FlushArgs {
    void *B;                      // TB [nw][nel][ld] (double, or float: fp32-stored inverse, R:A19)
    int nel, ld, np, K;
    int rows_per_cta;             // multiple of 8 * NG
    const int *win_count;
    const int *win_iel;
    const int *win_slot;          // [nw][K] slot of accepted move l in win_rows / vec
    const float *vec;             // orbital vector of (walker w, slot s) at vec + w * vec_wstride + s * vec_sstride
    size_t vec_wstride, vec_sstride;
    const double *win_rows;       // [nw][K][ld] R'[l] = (S^-T Rows)[l], accepted order
};

// Shared-memory geometry of one CTA, which owns LDC = ld / CS columns (strides chosen so every
// fragment load is bank-conflict free):
//   rows_s  double [KPAD][LDC + 4]  B-fragment of step 2: lane (g,t) reads row 4kq+t, column n0+g
//   v_s     float  [KPAD][LDC + 8]  B-fragment of step 1: lane (g,t) reads row 8nt+g, columns n0+2t,+1
//   part_s  double [PB][NG][NWC][8][KPAD + 4]   partial Q of each column warp (CS == 1: by block parity)
//   cpart_s double [2][8][KPAD + 4]             CS > 1: this CTA's partial Q, read by its cluster peers
//   kl_s    int [KPAD],  mbar
template <int KPAD, int LDC, int NWC, int NG, int CS>
struct FlushSmem {
    static constexpr int RS = LDC + 4, VS = LDC + 8, PS = KPAD + 4;
    static constexpr size_t rows_off = 0;
    static constexpr size_t v_off = rows_off + (size_t)KPAD * RS * sizeof(double);
    static constexpr size_t part_off = v_off + (size_t)KPAD * VS * sizeof(float);
    static constexpr size_t part_bytes = (size_t)NG * NWC * 8 * PS * sizeof(double);
    static constexpr size_t cpart_bytes = CS > 1 ? (size_t)2 * 8 * PS * sizeof(double) : 0;
    // CS == 1: two partial buffers (by block parity) save a barrier per block; one when shared
    // memory is short.  CS > 1: the cluster barrier of every block already orders their reuse.
    static constexpr int PB =
        (CS == 1 && part_off + 2 * part_bytes + KPAD * sizeof(int) + 16 <= 227 * 1024) ? 2 : 1;
    static constexpr size_t cpart_off = part_off + PB * part_bytes;
    static constexpr size_t kl_off = cpart_off + cpart_bytes;
    static constexpr size_t mbar_off = kl_off + (size_t)KPAD * sizeof(int);
    static constexpr size_t bytes = mbar_off + 16;
};

constexpr size_t kSmemMax = 227 * 1024;

// Row-block loop of the flush for a window of NTA active 8-wide tiles (8 NTA - 7 <= p <= 8 NTA): a
// compile-time count keeps the DMMA sequences free of branches, so the shared-memory operand loads
// and the fp32 -> fp64 conversions are scheduled ahead of the tensor-core instructions.
template <typename TB, int KPAD, int NWC, int TW, int NG, bool PF, int CS, int NTA>
__device__ __forceinline__ void flush_stream(const FlushArgs &a, int w, const double *rows_s, const float *v_s,
                                             double *part_s, double *cpart_s, const int *kl_s, uint64_t *mbar,
                                             int crank, int colbase)
{
    constexpr int LDC = NWC * TW * 8;
    constexpr int LD = LDC * CS;
    using L = FlushSmem<KPAD, LDC, NWC, NG, CS>;
    constexpr int RS = L::RS, VS = L::VS, PS = L::PS;
    constexpr int NTHREADS = 32 * NWC * NG;
    constexpr int KQA = 2 * NTA;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int grp = warp / NWC, wc = warp % NWC;
    const int nel = a.nel;

    // group `grp` takes blocks grp, grp + NG, ... of this CTA's rows.  With PF the next block's rows
    // are requested before the current block is contracted, so the HBM stream (loads of block i+1,
    // stores of block i-1) runs under the DMMA work of block i.
    const int m_begin = (blockIdx.x / CS) * a.rows_per_cta;
    const int m_end = min(nel, m_begin + a.rows_per_cta);
    const int col0 = 8 * TW * wc;                                  // within the CTA's slice
    TB *const walker_B = reinterpret_cast<TB *>(a.B) + (size_t)w * nel * LD + colbase + col0 + 2 * t;
    const float *const vfrag = v_s + g * VS + col0 + 2 * t;        // step-1 B fragments of this lane
    const double *const rfrag = rows_s + t * RS + col0 + g;        // step-2 B fragments of this lane
    bool staged = false;
    int m0 = m_begin + 8 * grp;
    double2 r[TW], rn[PF ? TW : 1];
    if (m0 < m_end) {
        const TB *src = walker_B + (size_t)min(m0 + g, nel - 1) * LD;
#pragma unroll
        for (int i = 0; i < TW; ++i) r[i] = ld2(src + 8 * i);
    }
    for (int it = 0; m0 < m_end; m0 += 8 * NG, ++it) {
        const int m = m0 + g;
        const int m0n = m0 + 8 * NG;
        if (PF && m0n < m_end) {
            const TB *src = walker_B + (size_t)min(m0n + g, nel - 1) * LD;
#pragma unroll
            for (int i = 0; i < TW; ++i) rn[PF ? i : 0] = ld2(src + 8 * i);
        }
        if (!staged) {
            mbar_wait(mbar, 0);
            staged = true;
        }
        // step 1: partial Q over this warp's columns
        double cq[NTA][2];
#pragma unroll
        for (int nt = 0; nt < NTA; ++nt) cq[nt][0] = cq[nt][1] = 0.0;
#pragma unroll
        for (int i = 0; i < TW; ++i) {
#pragma unroll
            for (int nt = 0; nt < NTA; ++nt) {
                const float2 f = *reinterpret_cast<const float2 *>(vfrag + 8 * nt * VS + 8 * i);
                dmma884(cq[nt][0], cq[nt][1], r[i].x, (double)f.x);
                dmma884(cq[nt][0], cq[nt][1], r[i].y, (double)f.y);
            }
        }
        // CS == 1: partials are double-buffered by block parity, one barrier per block is enough
        double *pbuf = part_s + (size_t)((L::PB == 2 ? (it & 1) : 0) * NG + grp) * NWC * 8 * PS;
        double *ps = pbuf + ((size_t)wc * 8 + g) * PS;
#pragma unroll
        for (int nt = 0; nt < NTA; ++nt)
            *reinterpret_cast<double2 *>(ps + 8 * nt + 2 * t) = make_double2(cq[nt][0], cq[nt][1]);
        // Q as A fragments: lane (g,t), k-step kq holds Q[m0+g][4kq+t], summed over the column slices
        double qa[KQA];
        if constexpr (CS == 1) {
            group_sync(1 + grp, 32 * NWC);
#pragma unroll
            for (int kq = 0; kq < KQA; ++kq) {
                const double *pp = pbuf + (size_t)g * PS + 4 * kq + t;
                double s = 0.0;
#pragma unroll
                for (int c = 0; c < NWC; ++c) s += pp[(size_t)c * 8 * PS];
                if (kl_s[4 * kq + t] == m) s -= 1.0;
                qa[kq] = s;
            }
            if (L::PB == 1) group_sync(1 + grp, 32 * NWC);
        } else {
            // two levels: this CTA's column warps first (fixed order), then the CTAs of the cluster
            // through distributed shared memory (fixed order: every CTA forms bit-identical Q)
            __syncthreads();
            double *cp = cpart_s + (size_t)(it & 1) * 8 * PS;
            for (int e = tid; e < 8 * 8 * NTA; e += NTHREADS) {
                const int row = e / (8 * NTA), col = e % (8 * NTA);
                double s = 0.0;
#pragma unroll
                for (int c = 0; c < NWC; ++c) s += pbuf[((size_t)c * 8 + row) * PS + col];
                cp[row * PS + col] = s;
            }
            cluster_arrive();
            cluster_wait();
#pragma unroll
            for (int kq = 0; kq < KQA; ++kq) {
                const double *pp = cp + (size_t)g * PS + 4 * kq + t;
                double s = 0.0;
#pragma unroll
                for (int c = 0; c < CS; ++c) s += (c == crank) ? *pp : ld_dsmem(pp, (uint32_t)c);
                if (kl_s[4 * kq + t] == m) s -= 1.0;
                qa[kq] = s;
            }
        }
        // step 2: B block -= Q R'; contraction index l = 4kq + t
#pragma unroll
        for (int kq = 0; kq < KQA; ++kq) {
            const double af = -qa[kq];
#pragma unroll
            for (int i = 0; i < TW; ++i) dmma884(r[i].x, r[i].y, af, rfrag[4 * kq * RS + 8 * i]);
        }
        if (m < nel) {
            TB *dst = walker_B + (size_t)m * LD;
#pragma unroll
            for (int i = 0; i < TW; ++i) st2(dst + 8 * i, r[i]);
        }
        if (PF) {
#pragma unroll
            for (int i = 0; i < TW; ++i) r[i] = rn[PF ? i : 0];
        } else if (m0n < m_end) {
            const TB *src = walker_B + (size_t)min(m0n + g, nel - 1) * LD;
#pragma unroll
            for (int i = 0; i < TW; ++i) r[i] = ld2(src + 8 * i);
        }
    }
    if (!staged) mbar_wait(mbar, 0);            // never leave with bulk copies in flight
    if constexpr (CS > 1) {                     // ... nor while a peer may still read this CTA's partials
        cluster_arrive();
        cluster_wait();
    }
}

// NWC column warps x TW 8-column tiles per warp = the CTA's LDC columns; NG row groups per CTA
// (CS == 1 only); PF = prefetch the next row block into registers; CS = cluster size.
template <typename TB, int KPAD, int NWC, int TW, int NG, bool PF, int CS>
__global__ void __launch_bounds__(32 * NWC * NG,
                                  (2 * (FlushSmem<KPAD, NWC * TW * 8, NWC, NG, CS>::bytes + 1024) <= 228 * 1024 &&
                                   2 * 32 * NWC * NG <= 1024) ? 2 : 1)
flush_dmma_kernel(FlushArgs a)
{
    static_assert(CS == 1 || NG == 1, "a cluster exchanges partials with a cluster-wide barrier: one row group");
    constexpr int LDC = NWC * TW * 8;
    constexpr int LD = LDC * CS;
    constexpr int NT = KPAD / 8;
    using L = FlushSmem<KPAD, LDC, NWC, NG, CS>;
    constexpr int RS = L::RS, VS = L::VS;
    constexpr int NTHREADS = 32 * NWC * NG;
    extern __shared__ __align__(128) unsigned char smem_flush[];
    double *rows_s = reinterpret_cast<double *>(smem_flush + L::rows_off);
    float *v_s = reinterpret_cast<float *>(smem_flush + L::v_off);
    double *part_s = reinterpret_cast<double *>(smem_flush + L::part_off);
    double *cpart_s = reinterpret_cast<double *>(smem_flush + L::cpart_off);
    int *kl_s = reinterpret_cast<int *>(smem_flush + L::kl_off);
    uint64_t *mbar = reinterpret_cast<uint64_t *>(smem_flush + L::mbar_off);

    const int w = blockIdx.y;
    const int p = a.win_count[w];
    if (p == 0) return;                                            // the whole cluster leaves together
    const int p8 = (p + 7) & ~7;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int K = a.K;
    const int crank = CS > 1 ? (int)cluster_ctarank() : 0;
    const int colbase = crank * LDC;                               // first column this CTA owns
    const int nvec = max(0, min(a.np - colbase, LDC));             // its share of the vectors' np columns

    // ---- stage the window: zero what the bulk copies do not write, then TMA the rows in
    if (tid == 0) mbar_init(mbar, 1);
    for (int e = tid; e < p * (LDC - nvec); e += NTHREADS) {       // pad columns of the vectors
        const int l = e / (LDC - nvec), c = nvec + e % (LDC - nvec);
        v_s[l * VS + c] = 0.f;
    }
    for (int e = tid; e < (p8 - p) * LDC; e += NTHREADS) {         // rows p..p8-1 of the last tile
        const int l = p + e / LDC, c = e % LDC;
        v_s[l * VS + c] = 0.f;
        rows_s[l * RS + c] = 0.0;
    }
    if (tid < KPAD) kl_s[tid] = tid < p ? a.win_iel[(size_t)w * K + tid] : -1;
    __syncthreads();
    if (warp == 0) {
        if (lane == 0)
            mbar_arrive_expect_tx(mbar, (uint32_t)p * (uint32_t)(LDC * sizeof(double) + nvec * sizeof(float)));
        __syncwarp();
        const double *rows_g = a.win_rows + (size_t)w * K * LD + colbase;
        const float *v_g = a.vec + (size_t)w * a.vec_wstride + colbase;
        for (int l = lane; l < p; l += 32) {
            const int slot = a.win_slot[(size_t)w * K + l];
            bulk_g2s(rows_s + l * RS, rows_g + (size_t)l * LD, LDC * sizeof(double), mbar);
            if (nvec) bulk_g2s(v_s + l * VS, v_g + (size_t)slot * a.vec_sstride, nvec * sizeof(float), mbar);
        }
    }

    // ---- stream the row blocks with the tile count of this window
    switch (p8 / 8) {
    case 1: flush_stream<TB, KPAD, NWC, TW, NG, PF, CS, 1>(a, w, rows_s, v_s, part_s, cpart_s, kl_s, mbar, crank, colbase); break;
    case 2: if constexpr (NT >= 2) flush_stream<TB, KPAD, NWC, TW, NG, PF, CS, 2>(a, w, rows_s, v_s, part_s, cpart_s, kl_s, mbar, crank, colbase); break;
    case 3: if constexpr (NT >= 3) flush_stream<TB, KPAD, NWC, TW, NG, PF, CS, 3>(a, w, rows_s, v_s, part_s, cpart_s, kl_s, mbar, crank, colbase); break;
    case 4: if constexpr (NT >= 4) flush_stream<TB, KPAD, NWC, TW, NG, PF, CS, 4>(a, w, rows_s, v_s, part_s, cpart_s, kl_s, mbar, crank, colbase); break;
    }
}

// qmc_det_accept_update appended the raw rows B0[k_l] (row l) and kept S^-1: turn the rows into
// R' = S^-T Rows in place before the flush.  One block per walker.
template <int KMAX>
__global__ void __launch_bounds__(256) rprime_kernel(int ld, int K, const int *win_count, const double *win_sinv,
                                                     double *win_rows)
{
    constexpr int GS = KMAX + 1;
    __shared__ double sinv_s[KMAX * GS];
    __shared__ long long rowoff_s[KMAX];
    const int w = blockIdx.x, p = win_count[w];
    if (p == 0) return;
    for (int e = threadIdx.x; e < p * p; e += 256) sinv_s[(e / p) * GS + e % p] = win_sinv[(size_t)w * K * K + (e / p) * K + e % p];
    if (threadIdx.x < p) rowoff_s[threadIdx.x] = (long long)threadIdx.x * ld;
    __syncthreads();
    double *rows = win_rows + (size_t)w * K * ld;
    rprime_warp<KMAX, double>(sinv_s, GS, p, rows, rowoff_s, rows, ld, threadIdx.x >> 5, 8, threadIdx.x & 31);
}

__global__ void reset_window_kernel(int nw, int *win_count)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < nw) win_count[w] = 0;
}

// Launch shapes.  X(V, NWC, TW, NG, PF, CS): ld = 64 V doubles = CS * NWC * TW * 8.  Several shapes
// may serve one ld, in order of measured preference; the first whose window fits shared memory is
// used (a cluster shape stages only ld / CS columns per CTA, so it serves the larger ranks).
#define QMC_FLUSH_SHAPES(X) \
    X(1, 1, 8, 4, true, 1) X(2, 2, 8, 4, true, 1) X(3, 3, 8, 4, true, 1) X(4, 4, 8, 4, true, 1) X(6, 6, 8, 2, true, 1) \
    X(8, 8, 8, 2, true, 1) X(8, 8, 4, 1, true, 2) \
    X(12, 6, 16, 2, false, 1) X(12, 6, 8, 1, true, 2) \
    X(16, 8, 16, 2, false, 1) X(16, 8, 8, 1, true, 2) X(16, 8, 4, 1, true, 4) \
    X(24, 12, 16, 1, false, 1) X(24, 6, 8, 1, true, 4) \
    X(32, 16, 16, 1, false, 1) X(32, 8, 8, 1, true, 4) X(32, 8, 4, 1, true, 8)

struct FlushShape { int id, nwc, tw, ng, cs; };

static size_t flush_smem_bytes(int kpad, const FlushShape &s)
{
    const size_t ldc = (size_t)s.nwc * s.tw * 8, ps = kpad + 4;
    const size_t base = (size_t)kpad * (ldc + 4) * 8 + (size_t)kpad * (ldc + 8) * 4;
    const size_t part = (size_t)s.ng * s.nwc * 8 * ps * 8, tail = (size_t)kpad * 4 + 16;
    if (s.cs > 1) return base + part + 2 * 8 * ps * 8 + tail;
    return base + (base + 2 * part + tail <= kSmemMax ? 2 : 1) * part + tail;
}

// window ranks the flush kernel is instantiated for
static int kpad_of(int K) { return K <= 8 ? 8 : (K <= 16 ? 16 : 32); }

// Shape for ld = 64 v and window rank kpad; id < 0 if none fits.
static FlushShape flush_shape(int v, int kpad)
{
    static const struct { int v; FlushShape s; } table[] = {
#define X(V, NWC, TW, NG, PF, CS) {V, {0, NWC, TW, NG, CS}},
        QMC_FLUSH_SHAPES(X)
#undef X
    };
    const int n = (int)(sizeof(table) / sizeof(table[0]));
    const char *env = getenv("QMC_FLUSH_SHAPE");        // tests: force the nth shape of this ld
    const int forced = env ? atoi(env) : -1;
    FlushShape fit{-1, 0, 0, 0, 0};
    int nth = 0;
    for (int i = 0; i < n; ++i) {
        if (table[i].v != v) continue;
        FlushShape s = table[i].s;
        s.id = i;
        const size_t b = flush_smem_bytes(kpad, s);
        if (forced >= 0) {
            if (nth++ == forced && b <= kSmemMax) return s;
            continue;
        }
        if (b <= kSmemMax) return s;
    }
    return fit;
}

// Largest delay rank whose window fits the flush kernel's shared memory for this ld.
int delayed_max_rank(int ld)
{
    int best = 0;
    for (int K = 2; K <= QMC_MAX_DELAY; ++K)
        if (flush_ring_serves(ld, K) || flush_shape(ld / 64, kpad_of(K)).id >= 0) best = K;
    return best;
}

template <typename TB, int KPAD, int NWC, int TW, int NG, bool PF, int CS>
static cudaError_t launch_flush_t(const FlushArgs &a, int nw, cudaStream_t s)
{
    using L = FlushSmem<KPAD, NWC * TW * 8, NWC, NG, CS>;
    if constexpr (L::bytes > kSmemMax) {
        return cudaErrorInvalidValue;
    } else {
        auto kern = flush_dmma_kernel<TB, KPAD, NWC, TW, NG, PF, CS>;
        // the opt-in is per device, not per process: set it on every launch (a host-side table write)
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::bytes);
        if (e != cudaSuccess) return e;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(CS * ((a.nel + a.rows_per_cta - 1) / a.rows_per_cta), nw);
        cfg.blockDim = dim3(32 * NWC * NG);
        cfg.dynamicSmemBytes = L::bytes;
        cfg.stream = s;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = CS;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = CS > 1 ? 1 : 0;
        return cudaLaunchKernelEx(&cfg, kern, a);
    }
}

template <typename TB, int NWC, int TW, int NG, bool PF, int CS>
static cudaError_t launch_flush_k(const FlushArgs &a, int nw, cudaStream_t s)
{
    switch (kpad_of(a.K)) {
    case 8: return launch_flush_t<TB, 8, NWC, TW, NG, PF, CS>(a, nw, s);
    case 16: return launch_flush_t<TB, 16, NWC, TW, NG, PF, CS>(a, nw, s);
    case 32: return launch_flush_t<TB, 32, NWC, TW, NG, PF, CS>(a, nw, s);
    }
    return cudaErrorInvalidValue;
}

int delayed_flush(qmc_det *d, cudaStream_t s)
{
    if (!d->delay || d->host_pending == 0) return QMC_OK;
    FlushArgs a{};
    a.B = d->b32 ? (void *)d->Bf : (void *)d->B;
    a.nel = d->nel; a.ld = d->ld; a.np = d->np; a.K = d->delay;
    a.win_count = d->win_count; a.win_iel = d->win_iel; a.win_slot = d->win_slot;
    a.vec = d->win_vec; a.vec_wstride = d->win_vec_wstride; a.vec_sstride = d->win_vec_sstride;
    a.win_rows = d->win_rows;
    const bool ring = flush_ring_serves(d->ld, d->delay);
    const FlushShape sh = ring ? FlushShape{0, 1, 1, 1, 1} : flush_shape(d->ld / 64, kpad_of(d->delay));
    QMC_REQUIRE(sh.id >= 0, "qmc_det_flush: no kernel shape for ld=%d, rank %d", d->ld, d->delay);
    // rows per CTA: the window is staged once per CTA, so prefer long CTAs when the grid stays large
    a.rows_per_cta = ((long long)d->nw * d->nel >= 128LL * d->nsm * 8) ? 128 : 64;
    if (a.rows_per_cta % (8 * sh.ng)) a.rows_per_cta = 8 * sh.ng * ((a.rows_per_cta + 8 * sh.ng - 1) / (8 * sh.ng));
    cudaError_t e = cudaErrorInvalidValue;
    if (d->win_rows_raw) {
        if (a.K <= 8) rprime_kernel<8><<<d->nw, 256, 0, s>>>(d->ld, a.K, d->win_count, d->win_sinv, d->win_rows);
        else if (a.K <= 16) rprime_kernel<16><<<d->nw, 256, 0, s>>>(d->ld, a.K, d->win_count, d->win_sinv, d->win_rows);
        else rprime_kernel<32><<<d->nw, 256, 0, s>>>(d->ld, a.K, d->win_count, d->win_sinv, d->win_rows);
        QMC_LAUNCHED();
        d->win_rows_raw = 0;
    }
    prof_start(d, kProfDelayedFlush, s);
    if (ring) e = flush_ring_launch(d, s);
    int id = 0;
#define X(V, NWC, TW, NG, PF, CS) \
    if (!ring && sh.id == id++)                                                              \
        e = d->b32 ? launch_flush_k<float, NWC, TW, NG, PF, CS>(a, d->nw, s) : launch_flush_k<double, NWC, TW, NG, PF, CS>(a, d->nw, s);
    QMC_FLUSH_SHAPES(X)
#undef X
    prof_stop(d, s);
    count_launch();
    QMC_CUDA(e);
    reset_window_kernel<<<(d->nw + 127) / 128, 128, 0, s>>>(d->nw, d->win_count);
    QMC_LAUNCHED();
    d->host_pending = 0;
    return QMC_OK;
}

}  // namespace qmc
