// Delayed (rank-k) update of the inverse (ref [44]; DESIGN.md R:O7).
#pragma once
#include "common.cuh"

namespace qmc {

int delayed_ratio(qmc_det *d, int iel, const float *phi, int ldo, double *ratio, cudaStream_t s);
int delayed_accept(qmc_det *d, int iel, const float *phi, int ldo, const double *ratio,
                   const unsigned char *accept, cudaStream_t s);
int delayed_flush(qmc_det *d, cudaStream_t s);
// One electron step of qmc_sweep in delayed mode (all pointers offset to the step).
int delayed_sweep_step(qmc_det *d, const qmc_spline *sp, double *pos, const double *delta, const double *unif,
                       int iel, double *ratios_out, unsigned char *accept_out, const unsigned char *forced,
                       float *phi_record, int nrecord, cudaStream_t s);

}  // namespace qmc
