// Flush of the delayed (rank-k) update for large N: the same two fp64 tensor-core contractions as
// flush.cu (DESIGN.md R:O7)
//
//     Q[m][l] = B0[m] . v_l - [k_l == m]           step 1
//     B[m]    = B0[m] - sum_l Q[m][l] * R'[l]       step 2,  R' = S^-T Rows
//
// in one pass over B, laid out for the B200 memory system:
//
//   * the walker's window lives in REGISTERS: warp wc of a CTA owns 8 TW columns and keeps the
//     step-1 fragments of v (converted to fp64 once) and the step-2 fragments of R' for those
//     columns, so the inner loops are pure DMMA.8x8x4 with no shared-memory operand traffic;
//   * the rows of B stream through a shared-memory RING filled by TMA bulk copies
//     (cp.async.bulk + mbarrier), several 8-row blocks ahead of the tensor cores, so the HBM read
//     stream never waits for a compute phase; results go back with 128-bit stores;
//   * a window of 16 rows x 1024 columns of (v, R') in fp64 is 256 KB -- a whole SM's register
//     file -- so the columns are split over a thread-block CLUSTER of CS CTAs; per row block every
//     CTA sends its 8 x p partial Q to its peers with st.async into their shared memory
//     (completion on the receiver's mbarrier: no fence, no cluster barrier);
//   * the loop is software-pipelined by one block: step 1 of block j is issued before step 2 of
//     block j-1, which hides the exchange latency behind tensor-core work.
//
// This file holds round 1's kernel (flush_ring_kernel: the reduction and exchange of the partial Q by two of
// the compute warps; QMC_FLUSH_LAG=0) and the dispatch of the ranks <= 16 to the warp-specialised kernel of
// flush_ring2.cuh, the default (the window fragments of 16 x 64 columns per warp fill the register file).
// Ranks 17..32 take flush_ring_hi.cu (the same kernel with 32 columns per warp) or flush_ring_hp.cu.  TB is the storage type of the inverse: double, or float
// for the single-precision inverse of PAPER.md L82 (R:A19) -- rows are converted when a fragment is
// loaded and rounded once when the block is stored; all arithmetic is fp64.
#include <stdlib.h>

#include "async_device.cuh"
#include "delayed_device.cuh"
#include "dmma.cuh"
#include "flush_ring2.cuh"

namespace qmc {


constexpr int kRecvBufs = 4;      // partial-Q receive buffers in flight (see the hazard note in the kernel)

// Shared memory of one CTA (LDC = NWC * TW * 8 columns):
//   ring   TB     [STAGES][8][LDC + 8]      row blocks of B (pitch + 8 elements: conflict-free vector reads)
//   part   double [2][NWC][8][KPAD + 4]     partial Q of each column warp, by block parity
//   recv   double [kRecvBufs][CS][8][KPAD + 4]   partial Q of every CTA of the cluster
//   full   mbarrier [STAGES], rbar mbarrier [kRecvBufs], pbar mbarrier [2]
template <typename TB, int KPAD, int TW, int NWC, int CS, int STAGES>
struct RingSmem {
    static constexpr int LDC = NWC * TW * 8, RP = LDC + 8, PS = KPAD + 4;
    static constexpr size_t ring_off = 0;
    static constexpr size_t part_off = ring_off + (size_t)STAGES * 8 * RP * sizeof(TB);
    static constexpr size_t recv_off = part_off + (size_t)2 * NWC * 8 * PS * sizeof(double);
    static constexpr size_t bar_off = recv_off + (size_t)kRecvBufs * CS * 8 * PS * sizeof(double);
    static constexpr size_t bytes = bar_off + (size_t)(STAGES + kRecvBufs + 2) * sizeof(uint64_t);
};

// Row-block loop for a window of NTA active 8-wide tiles (8 NTA - 7 <= p <= 8 NTA).
template <typename TB, int KPAD, int TW, int NWC, int CS, int STAGES, int NTA>
__device__ __forceinline__ void ring_stream(const RingArgs &a, int w, int p, unsigned char *smem)
{
    using L = RingSmem<TB, KPAD, TW, NWC, CS, STAGES>;
    constexpr int LDC = L::LDC, LD = LDC * CS, RP = L::RP, PS = L::PS;
    constexpr int KQA = 2 * NTA;
    constexpr int LW = NTA < NWC ? NTA : NWC;               // warps that reduce and send the partial Q
    // small clusters: the reducers run their own step 2 first (the other warps' partials are in by
    // then); larger clusters need the extra time for the exchange itself (measured both ways)
    constexpr bool SEND_LATE = CS <= 2;
    TB *ring = reinterpret_cast<TB *>(smem + L::ring_off);
    double *part = reinterpret_cast<double *>(smem + L::part_off);
    double *recv = reinterpret_cast<double *>(smem + L::recv_off);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + L::bar_off);
    uint64_t *rbar = full + STAGES;
    uint64_t *pbar = rbar + kRecvBufs;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int K = a.K, nel = a.nel;
    const uint32_t crank = CS > 1 ? cluster_ctarank() : 0u;
    const int colbase = (int)crank * LDC;                  // first column this CTA owns
    const int col0 = 8 * TW * warp;                        // this warp's first column within the slice

    // ---- the window, as DMMA B-fragments in registers
    double vf[TW][NTA][2], rf[TW][KQA];
    int klr[KQA];
#pragma unroll
    for (int nt = 0; nt < NTA; ++nt) {
        const int l = 8 * nt + g;
        const bool live = l < p;
        const float *vp = a.vec + (size_t)w * a.vec_wstride +
                          (live ? (size_t)a.win_slot[(size_t)w * K + l] * a.vec_sstride : 0);
#pragma unroll
        for (int i = 0; i < TW; ++i) {
            const int c = colbase + col0 + 8 * i + 2 * t;   // even; np is a multiple of 32
            float2 f = make_float2(0.f, 0.f);
            if (live && c < a.np) f = *reinterpret_cast<const float2 *>(vp + c);
            vf[i][nt][0] = (double)f.x;
            vf[i][nt][1] = (double)f.y;
        }
    }
#pragma unroll
    for (int kq = 0; kq < KQA; ++kq) {
        const int l = 4 * kq + t;
        const bool live = l < p;
        klr[kq] = live ? a.win_iel[(size_t)w * K + l] : -1;
        const double *rp = a.win_rows + ((size_t)w * K + (live ? l : 0)) * LD + colbase + col0 + g;
#pragma unroll
        for (int i = 0; i < TW; ++i) rf[i][kq] = live ? rp[8 * i] : 0.0;
    }

    // ---- the ring: warp 0 keeps STAGES - 1 row blocks in flight (starting it before the fragment
    // loads was measured: slower)
    const int m_begin = (blockIdx.x / CS) * a.rows_per_cta;
    const int m_end = min(nel, m_begin + a.rows_per_cta);
    const int nblk = (m_end - m_begin + 7) / 8;
    TB *const slice = reinterpret_cast<TB *>(a.B) + (size_t)w * nel * LD + colbase;     // row m of this CTA's slice at + m * LD
    auto issue = [&](int jb) {                                      // whole warp 0
        const int s = jb % STAGES, m0 = m_begin + 8 * jb, nv = min(8, m_end - m0);
        if (lane == 0) mbar_arrive_expect_tx(&full[s], (uint32_t)nv * (uint32_t)(LDC * sizeof(TB)));
        __syncwarp();
        if (lane < nv)
            bulk_g2s(ring + (size_t)(s * 8 + lane) * RP, slice + (size_t)(m0 + lane) * LD, LDC * sizeof(TB), &full[s]);
    };
    if (warp == 0)
        for (int jb = 0; jb < STAGES - 1 && jb < nblk; ++jb) issue(jb);

    // ---- software-pipelined loop: iteration j runs step 1 of block j and step 2 of block j - 1.
    // Hazards: ring stage (j-1) % STAGES is refilled by warp 0 at the top of iteration j; warp 0 is a
    // reducing warp, so in iteration j-1 it waited for every warp's partial of block j-1, which each
    // warp writes after reading that stage.  part[j & 1] is rewritten in iteration j+2, which a warp
    // reaches only after rbar of block j completed, i.e. after the reducers read part[j & 1].  A peer
    // sends block j+4 only after it received my block j+2, which I send after I read its block j
    // (iteration j+1): 4 receive buffers.
    double2 ra[TW], rb[TW];
    for (int j = 0; j <= nblk; ++j) {
        double *pbuf = part + (size_t)(j & 1) * NWC * 8 * PS;
        // the reducing warps: this CTA's partial (fixed order over its warps), sent to every CTA of the cluster
        auto reduce_and_send = [&]() {
            mbar_wait(&pbar[j & 1], (uint32_t)(j >> 1) & 1u);
            const int b = j % kRecvBufs;
            if (tid == 0) mbar_arrive_expect_tx(&rbar[b], (uint32_t)(CS * 64 * NTA * sizeof(double)));
            for (int e = tid; e < 64 * NTA; e += 32 * LW) {
                const int row = e / (8 * NTA), col = e % (8 * NTA);
                double sum = 0.0;
#pragma unroll
                for (int c = 0; c < NWC; ++c) sum += pbuf[((size_t)c * 8 + row) * PS + col];
                const double *dst = recv + ((size_t)(b * CS + (int)crank) * 8 + row) * PS + col;
#pragma unroll
                for (int c = 0; c < CS; ++c)
                    st_async_f64(mapa_u32(dst, (uint32_t)c), sum, mapa_u32(&rbar[b], (uint32_t)c));
            }
        };
        if (j < nblk) {
            if (warp == 0 && j + STAGES - 1 < nblk) issue(j + STAGES - 1);
            const int s = j % STAGES;
            mbar_wait(&full[s], (uint32_t)(j / STAGES) & 1u);
            const TB *src = ring + (size_t)(s * 8 + g) * RP + col0 + 2 * t;
#pragma unroll
            for (int i = 0; i < TW; ++i) rb[i] = ld2(src + 8 * i);
            // step 1: partial Q over this warp's columns
            double cq[NTA][2];
#pragma unroll
            for (int nt = 0; nt < NTA; ++nt) cq[nt][0] = cq[nt][1] = 0.0;
#pragma unroll
            for (int i = 0; i < TW; ++i)
#pragma unroll
                for (int nt = 0; nt < NTA; ++nt) {
                    dmma884(cq[nt][0], cq[nt][1], rb[i].x, vf[i][nt][0]);
                    dmma884(cq[nt][0], cq[nt][1], rb[i].y, vf[i][nt][1]);
                }
            double *ps = pbuf + ((size_t)warp * 8 + g) * PS;
#pragma unroll
            for (int nt = 0; nt < NTA; ++nt)
                *reinterpret_cast<double2 *>(ps + 8 * nt + 2 * t) = make_double2(cq[nt][0], cq[nt][1]);
            // hand the partial to the reducing warps through an mbarrier: the other warps do not stop
            // here (no CTA-wide barrier in the loop), so their DMMA work fills this exchange's bubbles
            __syncwarp();
            if (lane == 0) mbar_arrive(&pbar[j & 1]);
            if (!SEND_LATE && warp < LW) reduce_and_send();
        }
        if (j >= 1) {
            const int jj = j - 1, b = jj % kRecvBufs;
            const int m = m_begin + 8 * jj + g;
            mbar_wait(&rbar[b], (uint32_t)(jj / kRecvBufs) & 1u);
            // step 2: B block -= Q R'; Q read back in A-fragment layout, summed over the cluster in
            // a fixed order (every CTA forms bit-identical Q)
#pragma unroll
            for (int kq = 0; kq < KQA; ++kq) {
                const double *pp = recv + ((size_t)(b * CS) * 8 + g) * PS + 4 * kq + t;
                double q = 0.0;
#pragma unroll
                for (int c = 0; c < CS; ++c) q += pp[(size_t)c * 8 * PS];
                if (klr[kq] == m) q -= 1.0;
                const double af = -q;
#pragma unroll
                for (int i = 0; i < TW; ++i) dmma884(ra[i].x, ra[i].y, af, rf[i][kq]);
            }
            if (m < m_end) {
                TB *dst = slice + (size_t)m * LD + col0 + 2 * t;
#pragma unroll
                for (int i = 0; i < TW; ++i) st2(dst + 8 * i, ra[i]);
            }
        }
        if (SEND_LATE && j < nblk && warp < LW) reduce_and_send();
#pragma unroll
        for (int i = 0; i < TW; ++i) ra[i] = rb[i];
    }
}

template <typename TB, int KPAD, int TW, int NWC, int CS, int STAGES>
__global__ void __launch_bounds__(32 * NWC, 1) flush_ring_kernel(RingArgs a)
{
    using L = RingSmem<TB, KPAD, TW, NWC, CS, STAGES>;
    extern __shared__ __align__(128) unsigned char smem_ring[];
    const int w = blockIdx.y;
    const int p = a.win_count[w];
    if (p == 0) return;                                    // the whole cluster leaves together
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem_ring + L::bar_off);
    if (threadIdx.x == 0) {
        for (int i = 0; i < STAGES + kRecvBufs; ++i) mbar_init(&bars[i], 1);
        for (int i = 0; i < 2; ++i) mbar_init(&bars[STAGES + kRecvBufs + i], NWC);    // one arrival per warp
    }
    __syncthreads();
    if constexpr (CS > 1) {                                // peers' barriers exist before anything is sent
        cluster_arrive();
        cluster_wait();
    }
    constexpr int NT = KPAD / 8;
    switch ((p + 7) / 8) {
    case 1: ring_stream<TB, KPAD, TW, NWC, CS, STAGES, 1>(a, w, p, smem_ring); break;
    case 2: if constexpr (NT >= 2) ring_stream<TB, KPAD, TW, NWC, CS, STAGES, 2>(a, w, p, smem_ring); break;
    case 3: if constexpr (NT >= 3) ring_stream<TB, KPAD, TW, NWC, CS, STAGES, 3>(a, w, p, smem_ring); break;
    case 4: if constexpr (NT >= 4) ring_stream<TB, KPAD, TW, NWC, CS, STAGES, 4>(a, w, p, smem_ring); break;
    }
}

// Shapes: X(V, KPAD, TW, NWC, CS, STAGES) serves ld = 64 V = CS * NWC * TW * 8 and ranks <= KPAD.
#define QMC_RING_SHAPES(X) X(8, 16, 8, 8, 1, 5) X(16, 16, 8, 8, 2, 6) X(32, 16, 8, 8, 4, 5)

template <typename TB, int KPAD, int TW, int NWC, int CS, int STAGES>
static cudaError_t launch_ring(RingArgs a, int nw, int nsm, cudaStream_t s)
{
    // rows per CTA: the window fragments are loaded and the ring is filled once per CTA (a few us), so
    // prefer long CTAs as long as the grid still makes ~6 waves of one CTA per SM
    a.rows_per_cta = 64;
    for (int r = 1024; r >= 128; r >>= 1)
        if ((long long)nw * ((a.nel + r - 1) / r) * CS >= 6LL * nsm) { a.rows_per_cta = r; break; }
    using L = RingSmem<TB, KPAD, TW, NWC, CS, STAGES>;
    static_assert(L::bytes <= 227 * 1024, "ring shape exceeds shared memory");
    auto kern = flush_ring_kernel<TB, KPAD, TW, NWC, CS, STAGES>;
    // the opt-in is per device, not per process: set it on every launch (a host-side table write)
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::bytes);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(CS * ((a.nel + a.rows_per_cta - 1) / a.rows_per_cta), nw);
    cfg.blockDim = dim3(32 * NWC);
    cfg.dynamicSmemBytes = L::bytes;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CS;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;                                      // a 1-CTA cluster still addresses shared::cluster
    return cudaLaunchKernelEx(&cfg, kern, a);
}

// Shapes of the warp-specialised kernel: X(V, KPAD, TW, NWC, CS, ST1, ST2) serves ld = 64 V; ST1 = ring stages
// with LAG 1 (fp64 rows), ST2 = with LAG 2 (fp32 rows, half the bytes per stage).
#define QMC_RING2_SHAPES(X) X(8, 16, 8, 8, 1, 6, 10) X(16, 16, 8, 8, 2, 6, 10) X(32, 16, 8, 8, 4, 5, 9)

// Does a ring shape serve (ld, rank)?  QMC_FLUSH_RING=0 in the environment disables the ring kernels
// (A/B measurements and tests of the flush.cu kernel on the same shapes).
bool flush_ring_serves(int ld, int K)
{
    const char *env = getenv("QMC_FLUSH_RING");
    if ((env && atoi(env) == 0) || ld % 64) return false;
    if (K > 16) return flush_ring_hi_serves(ld, K) || flush_ring_hp_serves(ld, K);
    const int v = ld / 64;
#define X(V, KPAD, TW, NWC, CS, STAGES) \
    if (v == V) return true;
    QMC_RING_SHAPES(X)
#undef X
    return false;
}

// Enqueue the ring flush (the caller has checked flush_ring_serves and brackets it with its profiling events).
cudaError_t flush_ring_launch(qmc_det *d, cudaStream_t s)
{
    if (d->delay > 16) return flush_ring_hi_serves(d->ld, d->delay) ? flush_ring_hi_launch(d, s) : flush_ring_hp_launch(d, s);
    RingArgs a{};
    a.B = d->b32 ? (void *)d->Bf : (void *)d->B;
    a.nel = d->nel; a.ld = d->ld; a.np = d->np; a.K = d->delay;
    a.win_count = d->win_count; a.win_iel = d->win_iel; a.win_slot = d->win_slot;
    a.vec = d->win_vec; a.vec_wstride = d->win_vec_wstride; a.vec_sstride = d->win_vec_sstride;
    a.win_rows = d->win_rows;
    const int v = d->ld / 64;
    const char *lag = getenv("QMC_FLUSH_LAG");             // A/B hook, see below
    if (!(lag && atoi(lag) == 0)) {
        // QMC_FLUSH_LAG: 0 = the kernel above; 1 / 2 force the lag; QMC_FLUSH_PP: 1 = ping-pong on.
        // Default (measured on the B200 under its power cap, profiles/r02_flush_summary.md): lag 1 without
        // ping-pong for every shape and storage type -- 1.41 ms per flush at `large` (0.94 of the measured HBM
        // peak) against 1.55-1.59 ms for lag 2 with or without ping-pong and 1.62 ms for the round-1 kernel.
        const char *ppe = getenv("QMC_FLUSH_PP");
        const int lg = lag ? atoi(lag) : 1;
        const bool pp = ppe && atoi(ppe) == 1;
#define X(V, KPAD, TW, NWC, CS, ST1, ST2)                                                                           \
    if (v == V) {                                                                                                   \
        if (d->b32) {                                                                                               \
            if (lg == 2) return pp ? launch_ring2<true, 2, float, KPAD, TW, NWC, CS, ST2>(a, d->nw, d->nsm, s)      \
                                   : launch_ring2<false, 2, float, KPAD, TW, NWC, CS, ST2>(a, d->nw, d->nsm, s);    \
            return pp ? launch_ring2<true, 1, float, KPAD, TW, NWC, CS, ST2>(a, d->nw, d->nsm, s)                   \
                      : launch_ring2<false, 1, float, KPAD, TW, NWC, CS, ST2>(a, d->nw, d->nsm, s);                 \
        }                                                                                                           \
        if (lg == 2) return pp ? launch_ring2<true, 2, double, KPAD, TW, NWC, CS, ST1 - 1>(a, d->nw, d->nsm, s)     \
                               : launch_ring2<false, 2, double, KPAD, TW, NWC, CS, ST1 - 1>(a, d->nw, d->nsm, s);   \
        return pp ? launch_ring2<true, 1, double, KPAD, TW, NWC, CS, ST1>(a, d->nw, d->nsm, s)                      \
                  : launch_ring2<false, 1, double, KPAD, TW, NWC, CS, ST1>(a, d->nw, d->nsm, s);                    \
    }
        QMC_RING2_SHAPES(X)
#undef X
    }
#define X(V, KPAD, TW, NWC, CS, STAGES)                                                       \
    if (v == V)                                                                               \
        return d->b32 ? launch_ring<float, KPAD, TW, NWC, CS, STAGES>(a, d->nw, d->nsm, s)    \
                      : launch_ring<double, KPAD, TW, NWC, CS, STAGES>(a, d->nw, d->nsm, s);
    QMC_RING_SHAPES(X)
#undef X
    return cudaErrorInvalidValue;
}

}  // namespace qmc
