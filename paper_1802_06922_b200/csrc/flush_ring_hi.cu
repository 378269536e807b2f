// Ranks 17..32 of the delayed update on the warp-specialised ring flush kernel (flush_ring2.cuh; PAPER.md L112,
// L299; DESIGN.md R:O7): a window of 24 / 32 rows needs twice the fragment registers per column, so a compute
// warp owns 32 columns (TW = 4) and the columns of a row block are split over a cluster twice as wide as for
// ranks <= 16.  QMC_FLUSH_HP=1 in the environment routes these ranks to flush_ring_hp.cu instead (A/B hook).
#include <stdlib.h>

#include "flush_ring2.cuh"

namespace qmc {

// X(V, KPAD, TW, NWC, CS, A, B, C, D): ld = 64 V = CS * NWC * TW * 8; ring stages for fp64 rows / fp32 rows with
// LAG 1 (A, B: the default) and with LAG 2 (C, D: the A/B variant; 0 = does not fit, LAG 1 is used).
#define QMC_RING2_HI_SHAPES(X)                                                                        \
    X(8, 24, 4, 8, 2, 11, 16, 9, 16) X(16, 24, 4, 8, 4, 10, 16, 8, 16) X(32, 24, 4, 8, 8, 8, 16, 6, 12)  \
    X(8, 32, 4, 8, 2, 10, 16, 8, 16) X(16, 32, 4, 8, 4, 9, 16, 7, 14) X(32, 32, 4, 8, 8, 7, 14, 0, 7)

bool flush_ring_hi_serves(int ld, int K)
{
    const char *env = getenv("QMC_FLUSH_HP");
    if ((env && atoi(env) == 1) || ld % 64 || K <= 16 || K > 32) return false;
    const int v = ld / 64, kpad = K <= 24 ? 24 : 32;
#define X(V, KPAD, TW, NWC, CS, A, B, C, D) \
    if (v == V && kpad == KPAD) return true;
    QMC_RING2_HI_SHAPES(X)
#undef X
    return false;
}

cudaError_t flush_ring_hi_launch(qmc_det *d, cudaStream_t s)
{
    RingArgs a{};
    a.B = d->b32 ? (void *)d->Bf : (void *)d->B;
    a.nel = d->nel; a.ld = d->ld; a.np = d->np; a.K = d->delay;
    a.win_count = d->win_count; a.win_iel = d->win_iel; a.win_slot = d->win_slot;
    a.vec = d->win_vec; a.vec_wstride = d->win_vec_wstride; a.vec_sstride = d->win_vec_sstride;
    a.win_rows = d->win_rows;
    const int v = d->ld / 64, kpad = d->delay <= 24 ? 24 : 32;
    // QMC_FLUSH_LAG=2 / QMC_FLUSH_PP=1: the lag-2 and ping-pong variants (A/B hooks, as in flush_ring.cu)
    const char *lag = getenv("QMC_FLUSH_LAG"), *ppe = getenv("QMC_FLUSH_PP");
    const bool l2 = lag && atoi(lag) == 2, pp = ppe && atoi(ppe) == 1;
#define X(V, KPAD, TW, NWC, CS, A, B, C, D)                                                                             \
    if (v == V && kpad == KPAD) {                                                                                       \
        if constexpr (C > 0) {                                                                                          \
            if (l2 && pp) return d->b32 ? launch_ring2<true, 2, float, KPAD, TW, NWC, CS, D>(a, d->nw, d->nsm, s)        \
                                        : launch_ring2<true, 2, double, KPAD, TW, NWC, CS, C>(a, d->nw, d->nsm, s);      \
            if (l2) return d->b32 ? launch_ring2<false, 2, float, KPAD, TW, NWC, CS, D>(a, d->nw, d->nsm, s)            \
                                  : launch_ring2<false, 2, double, KPAD, TW, NWC, CS, C>(a, d->nw, d->nsm, s);          \
        }                                                                                                               \
        return d->b32 ? launch_ring2<false, 1, float, KPAD, TW, NWC, CS, B>(a, d->nw, d->nsm, s)                        \
                      : launch_ring2<false, 1, double, KPAD, TW, NWC, CS, A>(a, d->nw, d->nsm, s);                      \
    }
    QMC_RING2_HI_SHAPES(X)
#undef X
    return cudaErrorInvalidValue;
}

}  // namespace qmc
