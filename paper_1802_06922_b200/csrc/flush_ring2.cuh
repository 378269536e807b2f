// The warp-specialised ring flush kernel of the delayed update (DESIGN.md R:O7), shared by
// flush_ring.cu (ranks <= 16: 64 columns per compute warp) and flush_ring_hi.cu (ranks 17..32: 32 columns per
// compute warp).  See flush_ring.cu for the two contractions and the memory layout.
#pragma once
#include "async_device.cuh"
#include "delayed_device.cuh"
#include "dmma.cuh"

namespace qmc {

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

// ---------------------------------------------------------------------------------------------
// Warp-specialised ring flush (the default).  ncu of round 1's kernel (flush_ring.cu; profiles/r02_flush_summary.md):
// every warp spent 18 % of its time spinning on rbar.  There the partial Q of block j is reduced and sent by two
// of the COMPUTE warps, after their own step 2 of block j-1, which leaves the exchange one step 1 (~500
// cycles of DMMA) to complete -- not enough for reduce + st.async + arrival -- and all warps wait for the
// same event, so nothing fills the fp64 pipe meanwhile.  Here:
//   * a SERVICE warpgroup (4 warps, setmaxnreg hands their spare registers to the compute warps) feeds the
//     ring (TMA bulk copies) and reduces / sends the partial Q of a block the moment the last compute warp has
//     stored its share: no DMMA work stands in front of either;
//   * LAG = 1 (the default for every shape and storage type): per iteration a compute warp runs step 1 of block
//     j, publishes its partial Q, THEN waits for the exchange of block j-1 and runs step 2 on the row block it
//     kept in registers; the exchange has step 2 of block j-2 and step 1 of block j (~1000+ cycles of DMMA) to
//     complete, and the ring keeps every stage for prefetch;
//   * LAG = 2 (A/B variant, QMC_FLUSH_LAG=2): step 2 runs two blocks behind step 1 and reads its rows again
//     from the ring (a stage goes back to the producer through an `empty` mbarrier; bulk L2 prefetches run
//     ahead of the shortened ring -- they cost 19 % extra DRAM reads, which is why LAG 1 does without);
//   * the number of k-steps of step 2 follows p exactly (KQA = ceil(p / 4), not 2 NTA), and the -[k_l == m]
//     term of Q is applied once by the service warps instead of by every warp in step 2;
//   * optionally (PP, QMC_FLUSH_PP=1) the two compute warps of an SM sub-partition take turns on the fp64 pipe.
template <int LAG, typename TB, int KPAD, int TW, int NWC, int CS, int STAGES>
struct Ring2Smem {
    static constexpr int LDC = NWC * TW * 8, RP = LDC + 8, PS = KPAD + 4;
    static constexpr int NPB = LAG + 1;               // partial-Q buffers (block % NPB)
    static constexpr int NRB = LAG == 1 ? 4 : 6;      // receive buffers (hazard note in ring_stream2)
    static constexpr size_t ring_off = 0;
    static constexpr size_t part_off = ring_off + (size_t)STAGES * 8 * RP * sizeof(TB);
    static constexpr size_t recv_off = part_off + (size_t)NPB * NWC * 8 * PS * sizeof(double);
    static constexpr size_t kl_off = recv_off + (size_t)NRB * CS * 8 * PS * sizeof(double);
    static constexpr size_t bar_off = kl_off + (size_t)KPAD * sizeof(int);
    static constexpr int nbar = 2 * STAGES + NRB + NPB;     // full, empty, rbar, pbar
    static constexpr size_t bytes = bar_off + (size_t)nbar * sizeof(uint64_t);
};

template <bool SERVICE, bool PP, int LAG, typename TB, int KPAD, int TW, int NWC, int CS, int STAGES, int NTA, int KQA>
__device__ __forceinline__ void ring_stream2(const RingArgs &a, int w, int p, unsigned char *smem)
{
    using L = Ring2Smem<LAG, TB, KPAD, TW, NWC, CS, STAGES>;
    constexpr int LDC = L::LDC, LD = LDC * CS, RP = L::RP, PS = L::PS, NPB = L::NPB, NRB = L::NRB;
    // row blocks the TMA producer runs ahead in shared memory: LAG 1 frees a stage once every compute warp
    // has loaded it for step 1; LAG 2 keeps it until step 2 has read it again
    constexpr int PF = LAG == 1 ? STAGES - 1 : STAGES - 3;
    // ... and further ahead in L2 (bulk prefetch): only where the ring itself is short (LAG 2 keeps three stages
    // busy); with the deep LAG-1 ring the prefetches only add DRAM reads (ncu: +19 % read traffic)
    constexpr int kL2Ahead = LAG == 2 ? 4 : 0;
    static_assert(PF >= 1, "ring too short");
    TB *ring = reinterpret_cast<TB *>(smem + L::ring_off);
    double *part = reinterpret_cast<double *>(smem + L::part_off);
    double *recv = reinterpret_cast<double *>(smem + L::recv_off);
    const int *kl_s = reinterpret_cast<const int *>(smem + L::kl_off);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + L::bar_off);
    uint64_t *empty = full + STAGES;
    uint64_t *rbar = empty + STAGES;
    uint64_t *pbar = rbar + NRB;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int K = a.K, nel = a.nel;
    const uint32_t crank = CS > 1 ? cluster_ctarank() : 0u;
    const int colbase = (int)crank * LDC;                  // first column this CTA owns
    const int m_begin = (blockIdx.x / CS) * a.rows_per_cta;
    const int m_end = min(nel, m_begin + a.rows_per_cta);
    const int nblk = (m_end - m_begin + 7) / 8;
    TB *const slice = reinterpret_cast<TB *>(a.B) + (size_t)w * nel * LD + colbase;     // row m of this CTA's slice at + m * LD

    if constexpr (SERVICE) {
        // ---- the SERVICE warpgroup.  Warp h = 0 feeds the ring; warps h < 2 NTA reduce: per row block, lane e
        // sums element e of the compute warps' partial Q in a fixed order, applies the Kronecker term (CTA 0)
        // and sends the result to every CTA of the cluster.
        auto issue = [&](int jb) {
            const int s = jb % STAGES, m0 = m_begin + 8 * jb, nv = min(8, m_end - m0);
            if (LAG == 2 && jb >= STAGES) mbar_wait(&empty[s], (uint32_t)(jb / STAGES - 1) & 1u);   // every compute warp re-read block jb - STAGES
            if (lane == 0) mbar_arrive_expect_tx(&full[s], (uint32_t)nv * (uint32_t)(LDC * sizeof(TB)));
            __syncwarp();
            if (lane < nv)
                bulk_g2s(ring + (size_t)(s * 8 + lane) * RP, slice + (size_t)(m0 + lane) * LD, LDC * sizeof(TB), &full[s]);
        };
        auto prefetch = [&](int jb) {
            const int m0 = m_begin + 8 * jb, nv = min(8, m_end - m0);
            if (lane < nv) bulk_prefetch_l2(slice + (size_t)(m0 + lane) * LD, LDC * sizeof(TB));
        };
        const int h = warp - NWC;
        if (h == 0) {
            for (int jb = 0; jb <= PF && jb < nblk; ++jb) issue(jb);
            if (kL2Ahead)
                for (int jb = PF + 1; jb <= PF + kL2Ahead && jb < nblk; ++jb) prefetch(jb);
        }
        constexpr int NE = 64 * NTA, EPL = (NE + 127) / 128;      // elements of a block's partial Q; per lane of the warpgroup
        if (32 * h >= NE) return;
        for (int j = 0; j < nblk; ++j) {
            // LAG 2: the stage of block j + PF was released by step 2 of block j - 3 (compute iteration j - 1)
            if (LAG == 2 && h == 0 && j >= 1) {
                if (kL2Ahead && j + PF + kL2Ahead < nblk) prefetch(j + PF + kL2Ahead);
                if (j + PF < nblk) issue(j + PF);
            }
            const double *pbuf = part + (size_t)(j % NPB) * NWC * 8 * PS;
            const int b = j % NRB;
            if (h == 0 && lane == 0) mbar_arrive_expect_tx(&rbar[b], (uint32_t)(CS * NE * sizeof(double)));
            mbar_wait(&pbar[j % NPB], (uint32_t)(j / NPB) & 1u);
            // LAG 1: every compute warp has loaded block j for its step 1: the stage is free
            if (LAG == 1 && h == 0) {
                if (kL2Ahead && j + 1 + PF + kL2Ahead < nblk) prefetch(j + 1 + PF + kL2Ahead);
                if (j + 1 + PF < nblk) issue(j + 1 + PF);
            }
#pragma unroll
            for (int r = 0; r < EPL; ++r) {
                const int e = lane + 32 * h + 128 * r;
                if (e >= NE) break;
                const int row = e / (8 * NTA), col = e % (8 * NTA);
                double v[NWC];
#pragma unroll
                for (int c = 0; c < NWC; ++c) v[c] = pbuf[((size_t)c * 8 + row) * PS + col];
                double sum = v[0];
#pragma unroll
                for (int c = 1; c < NWC; ++c) sum += v[c];
                if (crank == 0 && kl_s[col] == m_begin + 8 * j + row) sum -= 1.0;
                const double *dst = recv + ((size_t)(b * CS + (int)crank) * 8 + row) * PS + col;
#pragma unroll
                for (int c = 0; c < CS; ++c)
                    st_async_f64(mapa_u32(dst, (uint32_t)c), sum, mapa_u32(&rbar[b], (uint32_t)c));
            }
        }
        return;
    } else {

    // ---- the COMPUTE warps.  The window, as DMMA B-fragments in registers:
    const int col0 = 8 * TW * warp;                        // this warp's first column within the slice
    double vf[TW][NTA][2], rf[TW][KQA];
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
        const double *rp = a.win_rows + ((size_t)w * K + (live ? l : 0)) * LD + colbase + col0 + g;
#pragma unroll
        for (int i = 0; i < TW; ++i) rf[i][kq] = live ? rp[8 * i] : 0.0;
    }

    // Iteration j: step 1 of block j, step 2 of block j - LAG.
    // Hazards.  part[j % NPB] is rewritten in iteration j + LAG + 1, which a warp reaches only after rbar of
    // block j completed (its step 2 in iteration j + LAG), i.e. after the service warps read it.  A CTA sends
    // block b' once all its compute warps finished step 1 of b', which they start only after the rbar wait of
    // block b' - LAG - 1 (step 2 in iteration b' - 1), i.e. after every compute warp of every CTA finished step
    // 1 of block b' - LAG - 1; a warp that still reads recv of block x (iteration x + LAG) has not started
    // step 1 of block x + LAG + 1, so b' <= x + 2 LAG + 1: 4 (LAG 1) / 6 (LAG 2) receive buffers.  LAG 1: ring
    // stage j % STAGES is refilled after pbar of block j (all compute warps loaded it); LAG 2: after all NWC
    // compute warps arrived on empty[] behind their step-2 reads.
    // PING-PONG (PP): warps r and r + 4 share an SM sub-partition and its fp64 pipe.  The barriers keep all
    // compute warps in step, so left alone both issue their DMMAs at the same time (each at half rate) and then
    // both do their loads, stores and barrier traffic while the pipe idles.  A token -- two named barriers
    // per pair -- makes them alternate: one issues the DMMAs of its iteration back to back (all operands
    // already in registers) while the other stores, signals and loads.
    const int pair = warp & 3, first = warp < 4;
    const int bar_mine = 1 + 2 * pair + (first ? 0 : 1), bar_other = 1 + 2 * pair + (first ? 1 : 0);
    if (PP && !first) named_arrive(bar_other, 64);         // the first warp of the pair starts
    double2 ra[TW];
    for (int j = 0; j < nblk + LAG; ++j) {
        const bool s1 = j < nblk, s2 = j >= LAG;
        const int jj = j - LAG, b = (jj + NRB) % NRB, sg1 = j % STAGES, sg2 = (jj + STAGES) % STAGES;
        double2 rb[TW];
        double qa[KQA];
        double cq[NTA][2];
        auto load1 = [&]() {                               // row block j from the ring
            mbar_wait(&full[sg1], (uint32_t)(j / STAGES) & 1u);
            const TB *src = ring + (size_t)(sg1 * 8 + g) * RP + col0 + 2 * t;
#pragma unroll
            for (int i = 0; i < TW; ++i) rb[i] = ld2(src + 8 * i);
        };
        auto load2 = [&]() {                               // row block j - LAG (LAG 2: again from the ring) and its Q
            if (LAG == 2) {
                const TB *src = ring + (size_t)(sg2 * 8 + g) * RP + col0 + 2 * t;
#pragma unroll
                for (int i = 0; i < TW; ++i) ra[i] = ld2(src + 8 * i);
            }
            mbar_wait(&rbar[b], (uint32_t)(jj / NRB) & 1u);
            // Q read back in A-fragment layout, summed over the cluster in a fixed order (every CTA forms
            // bit-identical Q)
#pragma unroll
            for (int kq = 0; kq < KQA; ++kq) {
                const double *pp = recv + ((size_t)(b * CS) * 8 + g) * PS + 4 * kq + t;
                double q = pp[0];
#pragma unroll
                for (int c = 1; c < CS; ++c) q += pp[(size_t)c * 8 * PS];
                qa[kq] = -q;
            }
        };
        auto step1 = [&]() {                               // partial Q over this warp's columns
#pragma unroll
            for (int nt = 0; nt < NTA; ++nt) cq[nt][0] = cq[nt][1] = 0.0;
#pragma unroll
            for (int i = 0; i < TW; ++i)
#pragma unroll
                for (int nt = 0; nt < NTA; ++nt) {
                    dmma884(cq[nt][0], cq[nt][1], rb[i].x, vf[i][nt][0]);
                    dmma884(cq[nt][0], cq[nt][1], rb[i].y, vf[i][nt][1]);
                }
        };
        auto step2 = [&]() {                               // B block -= Q R'
#pragma unroll
            for (int kq = 0; kq < KQA; ++kq)
#pragma unroll
                for (int i = 0; i < TW; ++i) dmma884(ra[i].x, ra[i].y, qa[kq], rf[i][kq]);
        };
        auto publish1 = [&]() {                            // hand the partial Q to the service warps
            double *ps = part + ((size_t)(j % NPB) * NWC * 8 + (size_t)warp * 8 + g) * PS;
#pragma unroll
            for (int nt = 0; nt < NTA; ++nt)
                *reinterpret_cast<double2 *>(ps + 8 * nt + 2 * t) = make_double2(cq[nt][0], cq[nt][1]);
            __syncwarp();
            if (lane == 0) mbar_arrive(&pbar[j % NPB]);
        };
        if (PP) {
            // all operands first, then the DMMAs of both steps back to back in this warp's turn
            if (s1) load1();
            if (s2) load2();
            named_sync(bar_mine, 64);                      // ---- my turn on the fp64 pipe
            if (s1) step1();
            if (s2) step2();
            named_arrive(bar_other, 64);                   // ---- the other warp's turn
            if (s1) publish1();
        } else {
            // step 1 first: the service warps reduce and send its result while this warp waits for the exchange
            // of block j - LAG, reads Q back and runs step 2
            if (s1) { load1(); step1(); publish1(); }
            if (s2) { load2(); step2(); }
        }
        if (s2) {
            if (LAG == 2) {
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[sg2]);   // this warp's reads of the stage are done (ra holds the block)
            }
            const int m = m_begin + 8 * jj + g;
            if (m < m_end) {
                TB *dst = slice + (size_t)m * LD + col0 + 2 * t;
#pragma unroll
                for (int i = 0; i < TW; ++i) st2(dst + 8 * i, ra[i]);
            }
        }
        if (LAG == 1) {
#pragma unroll
            for (int i = 0; i < TW; ++i) ra[i] = rb[i];
        }
    }
    if (PP && first) named_sync(bar_mine, 64);             // absorb the partner's last arrival
    }   // compute warps
}

template <bool PP, int LAG, typename TB, int KPAD, int TW, int NWC, int CS, int STAGES>
__global__ void __launch_bounds__(32 * (NWC + 4), 1) flush_ring2_kernel(RingArgs a)
{
    using L = Ring2Smem<LAG, TB, KPAD, TW, NWC, CS, STAGES>;
    extern __shared__ __align__(128) unsigned char smem_ring[];
    const int w = blockIdx.y;
    const int p = a.win_count[w];
    if (p == 0) return;                                    // the whole cluster leaves together
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem_ring + L::bar_off);
    int *kl_s = reinterpret_cast<int *>(smem_ring + L::kl_off);
    if (threadIdx.x < KPAD) kl_s[threadIdx.x] = (int)threadIdx.x < p ? a.win_iel[(size_t)w * a.K + threadIdx.x] : -1;
    if (threadIdx.x == 0) {
        for (int i = 0; i < STAGES; ++i) mbar_init(&bars[i], 1);                               // full: the producer's expect_tx
        for (int i = 0; i < STAGES; ++i) mbar_init(&bars[STAGES + i], NWC);                    // empty: one arrival per compute warp
        for (int i = 0; i < L::NRB; ++i) mbar_init(&bars[2 * STAGES + i], 1);                  // rbar
        for (int i = 0; i < L::NPB; ++i) mbar_init(&bars[2 * STAGES + L::NRB + i], NWC);       // pbar: one arrival per compute warp
    }
    __syncthreads();
    if constexpr (CS > 1) {                                // peers' barriers exist before anything is sent
        cluster_arrive();
        cluster_wait();
    }
    // The launch gives each of the 12 warps 168 registers; the service warpgroup needs few and hands the rest to
    // the two compute warpgroups, whose window fragments and row blocks need ~200-220.  The pool is the CTA's launch
    // allocation, 3 warpgroups x 168: 2 x 224 + 56 = 504 (asking for more would block the second warpgroup forever).
    constexpr int NT = KPAD / 8;
    const int kqa = (p + 3) / 4;                           // k-steps of step 2; NTA = ceil(KQA / 2)
    if ((int)(threadIdx.x >> 5) >= NWC) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        switch (kqa) {
        case 1: ring_stream2<true, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 1, 1>(a, w, p, smem_ring); break;
        case 2: ring_stream2<true, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 1, 2>(a, w, p, smem_ring); break;
        case 3: if constexpr (NT >= 2) ring_stream2<true, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 2, 3>(a, w, p, smem_ring); break;
        case 4: if constexpr (NT >= 2) ring_stream2<true, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 2, 4>(a, w, p, smem_ring); break;
        case 5: if constexpr (NT >= 3) ring_stream2<true, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 3, 5>(a, w, p, smem_ring); break;
        case 6: if constexpr (NT >= 3) ring_stream2<true, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 3, 6>(a, w, p, smem_ring); break;
        case 7: if constexpr (NT >= 4) ring_stream2<true, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 4, 7>(a, w, p, smem_ring); break;
        case 8: if constexpr (NT >= 4) ring_stream2<true, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 4, 8>(a, w, p, smem_ring); break;
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
    switch (kqa) {
    case 1: ring_stream2<false, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 1, 1>(a, w, p, smem_ring); break;
    case 2: ring_stream2<false, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 1, 2>(a, w, p, smem_ring); break;
    case 3: if constexpr (NT >= 2) ring_stream2<false, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 2, 3>(a, w, p, smem_ring); break;
    case 4: if constexpr (NT >= 2) ring_stream2<false, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 2, 4>(a, w, p, smem_ring); break;
    case 5: if constexpr (NT >= 3) ring_stream2<false, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 3, 5>(a, w, p, smem_ring); break;
    case 6: if constexpr (NT >= 3) ring_stream2<false, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 3, 6>(a, w, p, smem_ring); break;
    case 7: if constexpr (NT >= 4) ring_stream2<false, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 4, 7>(a, w, p, smem_ring); break;
    case 8: if constexpr (NT >= 4) ring_stream2<false, PP, LAG, TB, KPAD, TW, NWC, CS, STAGES, 4, 8>(a, w, p, smem_ring); break;
    }
    // (no barrier at the end: a CTA leaves after it has received every block its peers send it, and what it
    // sent lands in shared memory of CTAs that are still waiting for it)
}

template <bool PP, int LAG, typename TB, int KPAD, int TW, int NWC, int CS, int STAGES>
inline cudaError_t launch_ring2(RingArgs a, int nw, int nsm, cudaStream_t s)
{
    a.rows_per_cta = 64;
    for (int r = 1024; r >= 128; r >>= 1)
        if ((long long)nw * ((a.nel + r - 1) / r) * CS >= 6LL * nsm) { a.rows_per_cta = r; break; }
    using L = Ring2Smem<LAG, TB, KPAD, TW, NWC, CS, STAGES>;
    static_assert(L::bytes <= 227 * 1024, "ring shape exceeds shared memory");
    auto kern = flush_ring2_kernel<PP, LAG, TB, KPAD, TW, NWC, CS, STAGES>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::bytes);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(CS * ((a.nel + a.rows_per_cta - 1) / a.rows_per_cta), nw);
    cfg.blockDim = dim3(32 * (NWC + 4));       // 8 compute warps + the service warpgroup
    cfg.dynamicSmemBytes = L::bytes;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CS;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, a);
}


}  // namespace qmc
