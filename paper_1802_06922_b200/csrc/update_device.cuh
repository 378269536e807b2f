// Sherman-Morrison rank-1 update of B = (A^-1)^T in one pass (S4+S5 of the hot
// path).  Used by qmc_det_accept_update (decision given) and qmc_sweep (decision taken here from
// the ratio ratio_rowcopy_kernel left in d->ratio).
#pragma once
#include "common.cuh"

namespace qmc {

struct UpdateArgs {
    void *B;                      // TB [nw][nel][ld]
    int nel, ld, iel;
    const float *phi;             // [nw][ldphi] orbital vector of the proposal (fp32)
    size_t ldphi;                 //   walker stride in floats
    const double *rowk;           // [nw][ld] row iel of B before the update
    const double *ratio;          // [nw] det A'/det A of the proposal
    // decision given (qmc_det_accept_update)
    const unsigned char *accept;  // [nw]
    // decision taken here (qmc_sweep): all pointers already offset to (sweep, electron)
    const double *unif;           // [nw]
    const unsigned char *forced;  // [nw] or NULL
    int fixed_node;               // reject R < 0
    double *ratios_out;           // [nw] or NULL
    unsigned char *accept_out;    // [nw] or NULL
    double *pos;                  // [nw][nel][3]
    const double *delta;          // [nw][3]
    // drift moves (eq. 11-13): factor T(r'->r)/T(r->r') of the acceptance and the proposed positions
    const double *tfac;           // [nw] or NULL (= 1)
    const double *rprop;          // [nw][3] or NULL (the accepted electron moves to pos + delta)
    // per-walker statistics
    double *logdet;
    int *sign;
    long long *naccept;
};

constexpr int kUpdThreads = 256;
constexpr int kUpdRowsPerCta = 64;

// Metropolis test of eq. 12: accept iff R^2 tf > u, tf = 1 for symmetric T and a determinant-only Psi (R:A8),
// the ratio of the transition densities T'/T for drift moves, exp(-2 dJ) with a Jastrow factor.
__device__ __forceinline__ bool metropolis_t(double R, double tf, double u) { return isfinite(R) && isfinite(tf) && (R * R * tf > u); }
// A move may be applied only if its ratio is finite and non-zero: the update divides by R and the
// new Slater matrix would be singular otherwise (R:A18).  The Metropolis test already implies it
// (R * R > u >= 0); decisions imposed by the caller (forced_accept, qmc_det_accept_update) are
// filtered with it.
__device__ __forceinline__ bool usable_ratio(double R) { return isfinite(R) && R != 0.0; }

// One warp per row m: the row (ld = 64*VPT doubles) is read once into registers as VPT double2
// per lane, dotted with phi (warp-shuffle tree), updated with the old row iel, and written back:
// 16*ld bytes of HBM traffic per row (8*ld with the fp32-stored inverse), the floor for a rank-1 update.
template <typename TB, int VPT, bool DECIDE>
__global__ void __launch_bounds__(kUpdThreads) sm_update_kernel(UpdateArgs a)
{
    extern __shared__ double smem_upd[];
    const int w = blockIdx.y;
    const double R = a.ratio[w];
    bool acc;
    if (DECIDE) {
        const double tf = a.tfac ? a.tfac[w] : 1.0;
        acc = a.forced ? (a.forced[w] != 0) : (metropolis_t(R, tf, a.unif[w]) && !(a.fixed_node && R < 0.0));
    }
    else acc = a.accept[w] != 0;
    acc = acc && usable_ratio(R);     // an imposed accept of a singular / non-finite move is refused (R:A18)
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        if (DECIDE) {
            if (a.ratios_out) a.ratios_out[w] = R;
            if (a.accept_out) a.accept_out[w] = acc ? 1 : 0;
        }
        if (acc) {
            a.logdet[w] += log(fabs(R));
            if (R < 0.0) a.sign[w] = -a.sign[w];
            a.naccept[w] += 1;
            if (DECIDE) {
                double *r = a.pos + ((size_t)w * a.nel + a.iel) * 3;
                if (a.rprop) {
                    r[0] = a.rprop[3 * (size_t)w + 0]; r[1] = a.rprop[3 * (size_t)w + 1]; r[2] = a.rprop[3 * (size_t)w + 2];
                } else {
                    r[0] += a.delta[3 * (size_t)w + 0];
                    r[1] += a.delta[3 * (size_t)w + 1];
                    r[2] += a.delta[3 * (size_t)w + 2];
                }
            }
        }
    }
    if (!acc) return;

    const int ld = a.ld;
    double *phi_s = smem_upd;        // [ld]
    double *rowk_s = smem_upd + ld;  // [ld]
    const float *phi = a.phi + (size_t)w * a.ldphi;
    const double *rowk = a.rowk + (size_t)w * ld;
    for (int j = threadIdx.x; j < ld; j += kUpdThreads) {
        phi_s[j] = j < a.nel ? (double)phi[j] : 0.0;
        rowk_s[j] = rowk[j];
    }
    __syncthreads();

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int m_end = min(a.nel, (int)(blockIdx.x + 1) * kUpdRowsPerCta);
    const double2 *phi2 = reinterpret_cast<const double2 *>(phi_s);
    const double2 *rk2 = reinterpret_cast<const double2 *>(rowk_s);
    for (int m = blockIdx.x * kUpdRowsPerCta + wid; m < m_end; m += kUpdThreads / 32) {
        TB *row = reinterpret_cast<TB *>(a.B) + ((size_t)w * a.nel + m) * ld;
        double2 r[VPT];
#pragma unroll
        for (int i = 0; i < VPT; ++i) r[i] = ld2(row + 2 * (lane + 32 * i));
        double dot = 0.0;
#pragma unroll
        for (int i = 0; i < VPT; ++i) {
            const double2 p = phi2[lane + 32 * i];
            dot = fma(r[i].x, p.x, dot);
            dot = fma(r[i].y, p.y, dot);
        }
        dot = warp_sum(dot);
        const double f = (dot - (m == a.iel ? 1.0 : 0.0)) / R;
#pragma unroll
        for (int i = 0; i < VPT; ++i) {
            const double2 k2 = rk2[lane + 32 * i];
            r[i].x = fma(-f, k2.x, r[i].x);
            r[i].y = fma(-f, k2.y, r[i].y);
            st2(row + 2 * (lane + 32 * i), r[i]);
        }
    }
}

// ld (doubles) for nel electrons: a multiple of 64 whose quotient is one of the instantiated VPTs.
inline int update_ld(int nel)
{
    static const int vpts[] = {1, 2, 3, 4, 6, 8, 12, 16, 24, 32};
    const int need = (nel + 63) / 64;
    for (int v : vpts)
        if (v >= need) return 64 * v;
    return -1;
}

template <typename TB, bool DECIDE>
inline cudaError_t launch_sm_update(const UpdateArgs &a, int nw, cudaStream_t s)
{
    dim3 grid((a.nel + kUpdRowsPerCta - 1) / kUpdRowsPerCta, nw);
    const size_t smem = 2 * (size_t)a.ld * sizeof(double);
    switch (a.ld / 64) {
#define QMC_UPD_CASE(V)                                                              \
    case V:                                                                          \
        sm_update_kernel<TB, V, DECIDE><<<grid, kUpdThreads, smem, s>>>(a);              \
        break;
        QMC_UPD_CASE(1) QMC_UPD_CASE(2) QMC_UPD_CASE(3) QMC_UPD_CASE(4) QMC_UPD_CASE(6)
        QMC_UPD_CASE(8) QMC_UPD_CASE(12) QMC_UPD_CASE(16) QMC_UPD_CASE(24) QMC_UPD_CASE(32)
#undef QMC_UPD_CASE
    default:
        return cudaErrorInvalidValue;
    }
    count_launch();
    return cudaGetLastError();
}

}  // namespace qmc
