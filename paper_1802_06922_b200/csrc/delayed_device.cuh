// Delayed (rank-k) update of the inverse (ref [44]; DESIGN.md R:O7).
#pragma once
#include "common.cuh"

namespace qmc {

// SPO-VGL of electrons iel0 .. iel0+nb-1 of every walker at pos + delta (delta NULL: at pos) into `out`
// ([nb][nw][5][np], e.g. d->vgl) (sweep.cu); nb <= d->spo_batch.
int spo_batch_vgl(qmc_det *d, const qmc_spline *sp, const double *pos, const double *delta, int iel0, int nb,
                  float *phi_record, int nrecord, float *out, cudaStream_t s, bool per_walker_cursor = false);

int delayed_ratio(qmc_det *d, int iel, const float *phi, int ldo, double *ratio, cudaStream_t s);
int delayed_accept(qmc_det *d, int iel, const float *phi, int ldo, const double *ratio,
                   const unsigned char *accept, cudaStream_t s);
int delayed_flush(qmc_det *d, cudaStream_t s);
int delayed_flush_reset_host(qmc_det *d, cudaStream_t s);   // flush + forget the host-side window bookkeeping
bool flush_ring_serves(int ld, int K);                       // flush_ring.cu has a shape for (ld, rank)
cudaError_t flush_ring_launch(qmc_det *d, cudaStream_t s);    // enqueue it
bool flush_ring_hi_serves(int ld, int K);                    // flush_ring_hi.cu: the same for ranks 17..32
cudaError_t flush_ring_hi_launch(qmc_det *d, cudaStream_t s);
bool flush_ring_hp_serves(int ld, int K);                    // flush_ring_hp.cu: ranks 17..32, the earlier pipeline (A/B)
cudaError_t flush_ring_hp_launch(qmc_det *d, cudaStream_t s);
int delayed_max_rank(int ld);                                // largest K whose window fits shared memory
// One window of qmc_sweep in delayed mode: electrons iel0 .. iel0+nb-1 (nb <= delay rank), whose
// SPO-VGL is in d->vgl; ratios, decisions, moves and the flush.  Pointers are offset to the first step.
// fixed_node: reject R < 0; force_out: NULL or [nb][nw][3], F = 2 grad log Psi_T at the proposed configuration;
// record_mid: record d->ev_main on `s` between the window kernel and the flush (sweep.cu's second stream).
// jas: Jastrow factor of the window (base NULL = none): base[j][w] = dJ of step j against the configuration at
// the start of the window, corr[w][j][m] (m < j, row stride = the delay rank) = what an accepted step m adds to
// it (jastrow_move_kernel); the window kernel sums the pair terms of the steps it has accepted before step j
// and accepts iff R^2 exp(-2 dJ) > u.
struct WindowJastrow {
    const double *base;           // [nb][nw]
    const double *corr;           // [nw][ncorr][ncorr], ncorr = steps per window
    int ncorr;
    double *jratio_out;           // [nb][nw] or NULL: exp(-dJ)
};
int delayed_sweep_window(qmc_det *d, double *pos, const double *delta, const double *unif, int iel0, int nb,
                         double *ratios_out, unsigned char *accept_out, const unsigned char *forced,
                         int fixed_node, double *force_out, int record_mid, const WindowJastrow &jas, cudaStream_t s);

}  // namespace qmc
