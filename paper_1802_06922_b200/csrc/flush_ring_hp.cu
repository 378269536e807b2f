// Flush of the delayed (rank-k) update for large N and ranks 17..32: the two fp64 tensor-core
// contractions of flush_ring.cu (DESIGN.md R:O7)
//
//     Q[m][l] = B0[m] . v_l - [k_l == m]           step 1
//     B[m]    = B0[m] - sum_l Q[m][l] * R'[l]       step 2,  R' = S^-T Rows
//
// with the same building blocks (window fragments in registers, TMA ring, thread-block cluster with
// st.async exchange) in a pipeline made for the regime where the tensor pipe, not HBM, bounds the
// flush.  Per 8-row block a warp now owns 32 columns (the window of 24 / 32 rows needs the registers),
// so a block is half the tensor-core work of flush_ring.cu's and the reduce -> exchange -> reduce round
// trip can no longer hide behind one block (measured there: 1.8 us per block whatever the tile shape):
//
//   * WARP SPECIALISATION: 8 compute warps issue fragment loads, DMMAs and stores only; a warpgroup of 4
//     helper warps sums the partial Q over the compute warps (fixed order), sends it to the cluster,
//     sums what the cluster sent (fixed order: every CTA forms bit-identical Q), folds in the
//     -[k_l == m] term and leaves -Q in A-fragment order; helper 0 also feeds the ring.  setmaxnreg moves
//     the helpers' spare registers to the compute warpgroups (12 warps leave 168 each otherwise);
//   * step 2 runs kLag = 3 blocks behind step 1 (its rows are read again from the ring), so a compute
//     warp never waits for the exchange;
//   * PING-PONG: the two compute warps of an SM sub-partition pass a token (named barriers) and issue
//     their DMMAs in turn instead of at the same time.
// Measured on the B200 (profiles/r02_flush_summary.md): 0.55-0.6 of the fp64 tensor peak at rank 24 / 32
// against 0.41 for the rank-32 shapes of flush_ring.cu's pipeline; the ranks <= 16 stay with that
// kernel, which is the faster one per accepted move at N = 1024 and 2048.
//
// TB is the storage type of the inverse: double, or float for the single-precision inverse of
// PAPER.md L82 (R:A19) -- rows are converted when a fragment is loaded and rounded once when the
// block is stored; all arithmetic is fp64.
#include <stdlib.h>

#include "async_device.cuh"
#include "delayed_device.cuh"
#include "dmma.cuh"

namespace qmc {
namespace hp {

struct RingArgs {
    void *B;                      // TB [nw][nel][ld]
    int nel, ld, np, K;
    int rows_per_cta;             // multiple of 8
    const int *win_count;
    const int *win_iel;
    const int *win_slot;          // [nw][K] slot of accepted move l in vec
    const float *vec;             // orbital vector of (walker w, slot s) at vec + w * vec_wstride + s * vec_sstride
    size_t vec_wstride, vec_sstride;
    const double *win_rows;       // [nw][K][ld] R'[l], accepted order
};

constexpr int kLag = 3;           // step 2 runs this many blocks behind step 1
constexpr int kPartBufs = 3;      // partial-Q buffers of the compute warps   (hazards: see ring_compute)
constexpr int kRecvBufs = 6;      // partial-Q receive buffers
constexpr int kQBufs = 3;         // final -Q buffers

// Shared memory of one CTA (LDC = NWC * TW * 8 columns):
//   ring   TB     [STAGES][8][LDC + 8]           row blocks of B (pitch + 8 elements: conflict-free vector reads)
//   part   double [kPartBufs][NWC][8][KPAD + 4]  partial Q of each compute warp
//   recv   double [kRecvBufs][CS][8][KPAD + 4]   partial Q of every CTA of the cluster
//   qfin   double [kQBufs][8][KPAD + 4]          -(Q - [k_l == m]) summed over the cluster
//   kl     int    [KPAD]                         electron of accepted move l (-1 beyond p)
//   mbarriers: full[STAGES], empty[STAGES], pbar[kPartBufs], rbar[kRecvBufs], qbar[kQBufs]
template <typename TB, int KPAD, int TW, int NWC, int CS, int STAGES>
struct RingSmem {
    static constexpr int LDC = NWC * TW * 8, RP = LDC + 8, PS = KPAD + 4;
    static constexpr int NBAR = 2 * STAGES + kPartBufs + kRecvBufs + kQBufs;
    static constexpr size_t ring_off = 0;
    static constexpr size_t part_off = ring_off + (size_t)STAGES * 8 * RP * sizeof(TB);
    static constexpr size_t recv_off = part_off + (size_t)kPartBufs * NWC * 8 * PS * sizeof(double);
    static constexpr size_t qfin_off = recv_off + (size_t)kRecvBufs * CS * 8 * PS * sizeof(double);
    static constexpr size_t kl_off = qfin_off + (size_t)kQBufs * 8 * PS * sizeof(double);
    static constexpr size_t bar_off = kl_off + (size_t)KPAD * sizeof(int);
    static constexpr size_t bytes = bar_off + (size_t)NBAR * sizeof(uint64_t);
};

template <typename TB> struct RowVec;
template <> struct RowVec<double> {
    __device__ static __forceinline__ double2 load(const double *p) { return *reinterpret_cast<const double2 *>(p); }
    __device__ static __forceinline__ void store(double *p, double2 v) { *reinterpret_cast<double2 *>(p) = v; }
};
template <> struct RowVec<float> {
    __device__ static __forceinline__ double2 load(const float *p)
    {
        const float2 f = *reinterpret_cast<const float2 *>(p);
        return make_double2((double)f.x, (double)f.y);
    }
    __device__ static __forceinline__ void store(float *p, double2 v)
    {
        *reinterpret_cast<float2 *>(p) = make_float2((float)v.x, (float)v.y);     // round to nearest even, once
    }
};

template <typename TB, int KPAD, int TW, int NWC, int CS, int STAGES>
struct RingCtx {
    using L = RingSmem<TB, KPAD, TW, NWC, CS, STAGES>;
    TB *ring;
    double *part, *recv, *qfin;
    int *kl;
    uint64_t *full, *empty, *pbar, *rbar, *qbar;
    int m_begin, m_end, nblk;
    uint32_t crank;
    __device__ __forceinline__ RingCtx(unsigned char *smem, const RingArgs &a)
    {
        ring = reinterpret_cast<TB *>(smem + L::ring_off);
        part = reinterpret_cast<double *>(smem + L::part_off);
        recv = reinterpret_cast<double *>(smem + L::recv_off);
        qfin = reinterpret_cast<double *>(smem + L::qfin_off);
        kl = reinterpret_cast<int *>(smem + L::kl_off);
        full = reinterpret_cast<uint64_t *>(smem + L::bar_off);
        empty = full + STAGES;
        pbar = empty + STAGES;
        rbar = pbar + kPartBufs;
        qbar = rbar + kRecvBufs;
        crank = CS > 1 ? cluster_ctarank() : 0u;
        m_begin = (blockIdx.x / CS) * a.rows_per_cta;
        m_end = min(a.nel, m_begin + a.rows_per_cta);
        nblk = (m_end - m_begin + 7) / 8;
    }
};

constexpr int kHelpers = 4;       // helper warps per CTA (one warpgroup): reduction, exchange, ring producer

// A HELPER warp (h = 0..3) owns rows 2h, 2h + 1 of every 8-row block of partial Q.  Iteration i:
//   (1) when all compute warps have stored their partials of block i: sum them (pairwise tree: a fixed
//       order) and send the two rows to every CTA of the cluster (st.async);
//   (2) when the cluster's rows of block i - 1 have landed: sum them (ranks in order: every CTA forms
//       bit-identical Q), fold in -[k_l == m], store -Q for the compute warps;
//   (3) helper 0 refills the ring stage the compute warps released (step 2 runs kLag blocks behind).
// Its fp64 adds share the pipe with the compute warps' DMMAs and queue behind them (math-pipe
// throttle), which is why the work is spread over four warps and the compute warps run kLag blocks
// ahead: a helper has two block times for ~15 adds.
template <typename TB, int KPAD, int TW, int NWC, int CS, int STAGES, int NTA>
__device__ __forceinline__ void ring_helper(const RingArgs &a, int w, int h, const RingCtx<TB, KPAD, TW, NWC, CS, STAGES> &c)
{
    using L = RingSmem<TB, KPAD, TW, NWC, CS, STAGES>;
    constexpr int LDC = L::LDC, LD = LDC * CS, RP = L::RP, PS = L::PS;
    constexpr int N8 = 8 * NTA, NE = 2 * N8, EPL = (NE + 31) / 32;      // elements of my two rows; per lane
    static_assert(NWC == 8, "the reduction tree is written for 8 compute warps");
    const int lane = threadIdx.x & 31;
    const int nblk = c.nblk;
    int off[EPL], klane[EPL], rowl[EPL];
    bool live[EPL];
#pragma unroll
    for (int r = 0; r < EPL; ++r) {
        const int e = lane + 32 * r;
        live[r] = e < NE;
        const int row = 2 * h + (live[r] ? e / N8 : 0), col = live[r] ? e % N8 : 0;
        off[r] = row * PS + col;
        rowl[r] = row;
        klane[r] = c.kl[col];
    }
    const TB *slice = reinterpret_cast<const TB *>(a.B) + (size_t)w * a.nel * LD + (size_t)c.crank * LDC;
    int next = 0;                                          // next block to put into the ring (helper 0)
    auto produce = [&](int upto) {                         // issue blocks < upto whose stage is free
        for (; next < upto && next < nblk; ++next) {
            const int s = next % STAGES, m0 = c.m_begin + 8 * next, nv = min(8, c.m_end - m0);
            if (next >= STAGES) mbar_wait(&c.empty[s], (uint32_t)(next / STAGES + 1) & 1u);
            if (lane == 0) mbar_arrive_expect_tx(&c.full[s], (uint32_t)nv * (uint32_t)(LDC * sizeof(TB)));
            __syncwarp();
            if (lane < nv)
                bulk_g2s(c.ring + (size_t)(s * 8 + lane) * RP, slice + (size_t)(m0 + lane) * LD, LDC * sizeof(TB), &c.full[s]);
        }
    };
    if (h == 0) produce(STAGES);

    for (int i = 0; i <= nblk; ++i) {
        if (i < nblk) {                                   // (1) reduce over the compute warps, send
            const int b = i % kRecvBufs;
            mbar_wait(&c.pbar[i % kPartBufs], (uint32_t)(i / kPartBufs) & 1u);
            if (lane == 0) mbar_arrive_expect_tx(&c.rbar[b], (uint32_t)(CS * NE * sizeof(double)));
            const double *pbuf = c.part + (size_t)(i % kPartBufs) * NWC * 8 * PS;
            double v[EPL][NWC];
#pragma unroll
            for (int r = 0; r < EPL; ++r)
#pragma unroll
                for (int q = 0; q < NWC; ++q) v[r][q] = live[r] ? pbuf[(size_t)q * 8 * PS + off[r]] : 0.0;
            const uint32_t dst0 = smem_u32(c.recv + (size_t)(b * CS + (int)c.crank) * 8 * PS);
            const uint32_t bar0 = smem_u32(&c.rbar[b]);
#pragma unroll
            for (int r = 0; r < EPL; ++r) {
                const double sum = ((v[r][0] + v[r][1]) + (v[r][2] + v[r][3])) + ((v[r][4] + v[r][5]) + (v[r][6] + v[r][7]));
                if (live[r]) {
#pragma unroll
                    for (int q = 0; q < CS; ++q)
                        st_async_f64(mapa_addr(dst0 + (uint32_t)off[r] * 8u, (uint32_t)q), sum, mapa_addr(bar0, (uint32_t)q));
                }
            }
        }
        if (i >= 1) {                                     // (2) final -Q of block i - 1
            const int x = i - 1, b = x % kRecvBufs;
            mbar_wait(&c.rbar[b], (uint32_t)(x / kRecvBufs) & 1u);
            const double *src = c.recv + (size_t)(b * CS) * 8 * PS;
            double u[EPL][CS];
#pragma unroll
            for (int r = 0; r < EPL; ++r)
#pragma unroll
                for (int q = 0; q < CS; ++q) u[r][q] = live[r] ? src[(size_t)q * 8 * PS + off[r]] : 0.0;
            double *qf = c.qfin + (size_t)(x % kQBufs) * 8 * PS;
            const int m0 = c.m_begin + 8 * x;
#pragma unroll
            for (int r = 0; r < EPL; ++r) {
                double sum = u[r][0];
#pragma unroll
                for (int q = 1; q < CS; ++q) sum += u[r][q];
                if (klane[r] == m0 + rowl[r]) sum -= 1.0;
                if (live[r]) qf[off[r]] = -sum;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&c.qbar[x % kQBufs]);
        }
        if (h == 0) produce(i + 1 + STAGES - kLag);       // (3) stages released up to compute iteration i
    }
}

// A COMPUTE warp, for a window of NTA active 8-wide tiles (8 NTA - 7 <= p <= 8 NTA): iteration j runs
// step 1 of block j (partial Q over this warp's columns -> part[j % 3][warp]) and step 2 of block
// j - kLag (rows read again from the ring, -Q from the helpers), then releases that ring stage.
// Hazards.  part[j % 3] is rewritten in iteration j + 3, after the warp passed qbar of block j (top
// of iteration j + 3), which the helpers form after they reduced block j + 1.  qfin[x % 3] is rewritten for
// block x + 3 after pbar of block x + 4 completed, i.e. after every compute warp finished iteration
// x + 3 and with it step 2 of block x.  A peer's helper sends block x + 6 after its compute warps
// passed qbar of block x + 2, which needs my helper's send of block x + 2, issued an iteration after it
// read recv[x % 6].
template <typename TB, int KPAD, int TW, int NWC, int CS, int STAGES, int NTA>
__device__ __forceinline__ void ring_compute(const RingArgs &a, int w, int p, const RingCtx<TB, KPAD, TW, NWC, CS, STAGES> &c)
{
    using L = RingSmem<TB, KPAD, TW, NWC, CS, STAGES>;
    constexpr int LDC = L::LDC, LD = LDC * CS, RP = L::RP, PS = L::PS;
    constexpr int KQA = 2 * NTA;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int K = a.K;
    const int colbase = (int)c.crank * LDC;                // first column this CTA owns
    const int col0 = 8 * TW * warp;                        // this warp's first column within the slice

    // ---- the window, as DMMA B-fragments in registers
    double vf[TW][NTA][2], rf[TW][KQA];
#pragma unroll
    for (int nt = 0; nt < NTA; ++nt) {
        const int l = 8 * nt + g;
        const bool live = l < p;
        const float *vp = a.vec + (size_t)w * a.vec_wstride +
                          (live ? (size_t)a.win_slot[(size_t)w * K + l] * a.vec_sstride : 0);
#pragma unroll
        for (int i = 0; i < TW; ++i) {
            const int cc = colbase + col0 + 8 * i + 2 * t;  // even; np is a multiple of 32
            float2 f = make_float2(0.f, 0.f);
            if (live && cc < a.np) f = *reinterpret_cast<const float2 *>(vp + cc);
            vf[i][nt][0] = (double)f.x;
            vf[i][nt][1] = (double)f.y;
        }
    }
#pragma unroll
    for (int kq = 0; kq < KQA; ++kq) {
        const int l = 4 * kq + t;
        const bool live = l < p;
        const double *rp = a.win_rows + ((size_t)w * K + (live ? l : 0)) * LD + colbase + col0 + g;
#pragma unroll
        for (int i = 0; i < TW; ++i) rf[i][kq] = live ? rp[8 * i] : 0.0;
    }

    TB *const slice = reinterpret_cast<TB *>(a.B) + (size_t)w * a.nel * LD + colbase;   // row m of this CTA's slice at + m * LD
    const int nblk = c.nblk;
    // PING-PONG.  Warps r and r + 4 share an SM sub-partition and its tensor pipe.  The barriers keep all
    // compute warps in step, so left alone both would issue their DMMAs at the same time (each at half
    // rate) and then both do their loads, stores and barrier traffic while the pipe idles (measured:
    // 41 % idle).  A token -- two named barriers per pair -- makes them alternate instead: one issues
    // the 24 K DMMAs of its iteration back to back while the other does everything else.
    const int pair = warp & 3, first = warp < 4;
    const int bar_mine = 1 + 2 * pair + (first ? 0 : 1), bar_other = 1 + 2 * pair + (first ? 1 : 0);
    if (!first) named_arrive(bar_other, 64);               // the first warp of the pair starts
    for (int j = 0; j < nblk + kLag; ++j) {
        const bool s1 = j < nblk, s4 = j >= kLag;
        const int x = j - kLag;
        // -Q of block j - kLag first: once it is there the helpers are also done with part[j % 3]
        if (s4) mbar_wait(&c.qbar[x % kQBufs], (uint32_t)(x / kQBufs) & 1u);
        if (s1) mbar_wait(&c.full[j % STAGES], (uint32_t)(j / STAGES) & 1u);
        double2 rb[TW], ra[TW];
        double qa[KQA];
        if (s1) {
            const TB *src = c.ring + (size_t)((j % STAGES) * 8 + g) * RP + col0 + 2 * t;
#pragma unroll
            for (int i = 0; i < TW; ++i) rb[i] = RowVec<TB>::load(src + 8 * i);
        }
        named_sync(bar_mine, 64);   // ---- my turn on the tensor pipe
        if (s4) {                                          // (these loads land under the DMMAs of step 1)
            const TB *src = c.ring + (size_t)((x % STAGES) * 8 + g) * RP + col0 + 2 * t;
#pragma unroll
            for (int i = 0; i < TW; ++i) ra[i] = RowVec<TB>::load(src + 8 * i);
            const double *qf = c.qfin + ((size_t)(x % kQBufs) * 8 + g) * PS + t;
#pragma unroll
            for (int kq = 0; kq < KQA; ++kq) qa[kq] = qf[4 * kq];
        }
        // step 1 of block j: two accumulator sets per tile (even / odd k-steps), 2 NTA independent chains
        double cq[NTA][2], cr[NTA][2];
        if (s1) {
#pragma unroll
            for (int nt = 0; nt < NTA; ++nt) cq[nt][0] = cq[nt][1] = cr[nt][0] = cr[nt][1] = 0.0;
#pragma unroll
            for (int i = 0; i < TW; ++i)
#pragma unroll
                for (int nt = 0; nt < NTA; ++nt) {
                    dmma884(cq[nt][0], cq[nt][1], rb[i].x, vf[i][nt][0]);
                    dmma884(cr[nt][0], cr[nt][1], rb[i].y, vf[i][nt][1]);
                }
        }
        if (s4) {                                          // step 2 of block j - kLag
#pragma unroll
            for (int kq = 0; kq < KQA; ++kq) {
                if (4 * kq >= p) continue;                  // whole k-step beyond the window (warp-uniform)
#pragma unroll
                for (int i = 0; i < TW; ++i) dmma884(ra[i].x, ra[i].y, qa[kq], rf[i][kq]);
            }
        }
        named_arrive(bar_other, 64);   // ---- the other warp's turn
        if (s1) {
            double *ps = c.part + (((size_t)(j % kPartBufs) * NWC + warp) * 8 + g) * PS;
#pragma unroll
            for (int nt = 0; nt < NTA; ++nt)
                *reinterpret_cast<double2 *>(ps + 8 * nt + 2 * t) = make_double2(cq[nt][0] + cr[nt][0], cq[nt][1] + cr[nt][1]);
            __syncwarp();
            if (lane == 0) mbar_arrive(&c.pbar[j % kPartBufs]);
        }
        if (s4) {
            const int m = c.m_begin + 8 * x + g;
            if (m < c.m_end) {
                TB *dst = slice + (size_t)m * LD + col0 + 2 * t;
#pragma unroll
                for (int i = 0; i < TW; ++i) RowVec<TB>::store(dst + 8 * i, ra[i]);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&c.empty[x % STAGES]);
        }
    }
    if (first) named_sync(bar_mine, 64);   // absorb the partner's last arrival
}

template <typename TB, int KPAD, int TW, int NWC, int CS, int STAGES>
__global__ void __launch_bounds__(32 * (NWC + kHelpers), 1) flush_ring_kernel(RingArgs a)
{
    using L = RingSmem<TB, KPAD, TW, NWC, CS, STAGES>;
    extern __shared__ __align__(128) unsigned char smem_ring[];
    const int w = blockIdx.y;
    const int p = a.win_count[w];
    if (p == 0) return;                                    // the whole cluster leaves together
    RingCtx<TB, KPAD, TW, NWC, CS, STAGES> c(smem_ring, a);
    if (threadIdx.x == 0) {
        for (int i = 0; i < STAGES; ++i) { mbar_init(&c.full[i], 1); mbar_init(&c.empty[i], NWC); }
        for (int i = 0; i < kPartBufs; ++i) mbar_init(&c.pbar[i], NWC);       // one arrival per compute warp
        for (int i = 0; i < kRecvBufs; ++i) mbar_init(&c.rbar[i], kHelpers);  // one per helper (+ the bytes the cluster sends)
        for (int i = 0; i < kQBufs; ++i) mbar_init(&c.qbar[i], kHelpers);
    }
    if (threadIdx.x < KPAD) c.kl[threadIdx.x] = (int)threadIdx.x < p ? a.win_iel[(size_t)w * a.K + threadIdx.x] : -1;
    __syncthreads();
    if constexpr (CS > 1) {                                // peers' barriers exist before anything is sent
        cluster_arrive();
        cluster_wait();
    }
    const int nta = (p + 7) / 8;
    constexpr int NT = KPAD / 8;
    const int hw = (int)(threadIdx.x >> 5) - NWC;
    // The launch gives every warp 168 registers (12 warps, 3 per sub-partition).  The helper warpgroup
    // needs ~40 and hands the rest to the two compute warpgroups, whose window fragments need more.
    if (hw >= 0) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        switch (nta) {
        case 1: ring_helper<TB, KPAD, TW, NWC, CS, STAGES, 1>(a, w, hw, c); break;
        case 2: if constexpr (NT >= 2) ring_helper<TB, KPAD, TW, NWC, CS, STAGES, 2>(a, w, hw, c); break;
        case 3: if constexpr (NT >= 3) ring_helper<TB, KPAD, TW, NWC, CS, STAGES, 3>(a, w, hw, c); break;
        case 4: if constexpr (NT >= 4) ring_helper<TB, KPAD, TW, NWC, CS, STAGES, 4>(a, w, hw, c); break;
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
    switch (nta) {
    case 1: ring_compute<TB, KPAD, TW, NWC, CS, STAGES, 1>(a, w, p, c); break;
    case 2: if constexpr (NT >= 2) ring_compute<TB, KPAD, TW, NWC, CS, STAGES, 2>(a, w, p, c); break;
    case 3: if constexpr (NT >= 3) ring_compute<TB, KPAD, TW, NWC, CS, STAGES, 3>(a, w, p, c); break;
    case 4: if constexpr (NT >= 4) ring_compute<TB, KPAD, TW, NWC, CS, STAGES, 4>(a, w, p, c); break;
    }
}

// Shapes: X(V, KPAD, TW, NWC, CS, STAGES) serves ld = 64 V = CS * NWC * TW * 8 and ranks 17..KPAD
// (32 columns per compute warp; the ring as deep as shared memory allows).
#define QMC_RING_HP_SHAPES(X) \
    X(8, 24, 4, 8, 2, 9) X(16, 24, 4, 8, 4, 8) X(32, 24, 4, 8, 8, 5) \
    X(8, 32, 4, 8, 2, 8) X(16, 32, 4, 8, 4, 6)

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
    cfg.blockDim = dim3(32 * (NWC + kHelpers));
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

}  // namespace hp

// Does a shape of this kernel serve (ld, rank 17..32)?
bool flush_ring_hp_serves(int ld, int K)
{
    if (ld % 64 || K <= 16 || K > 32) return false;
    const int v = ld / 64, kpad = K <= 24 ? 24 : 32;
#define X(V, KPAD, TW, NWC, CS, STAGES) \
    if (v == V && kpad == KPAD) return true;
    QMC_RING_HP_SHAPES(X)
#undef X
    return false;
}

cudaError_t flush_ring_hp_launch(qmc_det *d, cudaStream_t s)
{
    hp::RingArgs a{};
    a.B = d->b32 ? (void *)d->Bf : (void *)d->B;
    a.nel = d->nel; a.ld = d->ld; a.np = d->np; a.K = d->delay;
    a.win_count = d->win_count; a.win_iel = d->win_iel; a.win_slot = d->win_slot;
    a.vec = d->win_vec; a.vec_wstride = d->win_vec_wstride; a.vec_sstride = d->win_vec_sstride;
    a.win_rows = d->win_rows;
    const int v = d->ld / 64, kpad = d->delay <= 24 ? 24 : 32;
#define X(V, KPAD, TW, NWC, CS, STAGES)                                                           \
    if (v == V && kpad == KPAD)                                                                   \
        return d->b32 ? hp::launch_ring<float, KPAD, TW, NWC, CS, STAGES>(a, d->nw, d->nsm, s)    \
                      : hp::launch_ring<double, KPAD, TW, NWC, CS, STAGES>(a, d->nw, d->nsm, s);
    QMC_RING_HP_SHAPES(X)
#undef X
    return cudaErrorInvalidValue;
}

}  // namespace qmc
