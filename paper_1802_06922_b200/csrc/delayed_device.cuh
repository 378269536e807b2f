// Delayed (rank-k) update of the inverse (ref [44]; DESIGN.md R:O7).
#pragma once
#include "common.cuh"

namespace qmc {

int delayed_ratio(qmc_det *d, int iel, const float *phi, int ldo, double *ratio, cudaStream_t s);
int delayed_accept(qmc_det *d, int iel, const float *phi, int ldo, const double *ratio,
                   const unsigned char *accept, cudaStream_t s);
int delayed_flush(qmc_det *d, cudaStream_t s);
int delayed_flush_reset_host(qmc_det *d, cudaStream_t s);   // flush + forget the host-side window bookkeeping
int delayed_max_rank(int ld);                                // largest K whose window fits shared memory
// SPO-VGL of every walker's proposal pos[w][iel] + delta[w] into d->vgl (sweep.cu)
int spo_proposal_vgl(qmc_det *d, const qmc_spline *sp, const double *pos, const double *delta, int iel,
                     float *phi_record, int nrecord, cudaStream_t s);
// One electron step of qmc_sweep in delayed mode (all pointers offset to the step).
int delayed_sweep_step(qmc_det *d, const qmc_spline *sp, double *pos, const double *delta, const double *unif,
                       int iel, double *ratios_out, unsigned char *accept_out, const unsigned char *forced,
                       float *phi_record, int nrecord, cudaStream_t s);

}  // namespace qmc
