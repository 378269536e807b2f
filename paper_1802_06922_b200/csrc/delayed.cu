// Delayed (rank-k) update -- placeholder until the rank-1 path is measured.
#include "delayed_device.cuh"

namespace qmc {

int delayed_ratio(qmc_det *, int, const float *, int, double *, cudaStream_t)
{
    set_error("delayed update: not implemented yet");
    return QMC_EINVAL;
}
int delayed_accept(qmc_det *, int, const float *, int, const double *, const unsigned char *, cudaStream_t)
{
    set_error("delayed update: not implemented yet");
    return QMC_EINVAL;
}
int delayed_flush(qmc_det *, cudaStream_t)
{
    set_error("delayed update: not implemented yet");
    return QMC_EINVAL;
}

int delayed_sweep_step(qmc_det *, const qmc_spline *, double *, const double *, const double *, int, double *,
                       unsigned char *, const unsigned char *, float *, int, cudaStream_t)
{
    set_error("delayed update: not implemented yet");
    return QMC_EINVAL;
}

}  // namespace qmc
