"""B200-native particle-by-particle QMC move (after arxiv 1802.06922): spline SPO-VGL,
determinant ratio, Sherman-Morrison / delayed update, sweep driver -- CUDA (sm_100a) behind a
C ABI (include/qmc_b200.h).  The CUDA library is loaded lazily by `api`; `inputs` needs no GPU."""
__all__ = ["api", "inputs", "build"]
