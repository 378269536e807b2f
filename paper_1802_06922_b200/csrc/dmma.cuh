// fp64 tensor-core building blocks shared by the delayed-update kernels (window.cu, flush.cu,
// delayed.cu): mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4) and the R' = S^-T Rows contraction.
#pragma once
#include "common.cuh"

namespace qmc {

// C (8x8) += A (8x4, row) * B (4x8, col).  Lane (g = lane / 4, t = lane % 4) holds A[g][t],
// B[t][g] and C[g][2t], C[g][2t+1].
__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// Flush operand of the delayed update (DESIGN.md R:O7): with T = Q S^-T, B -= T Rows = Q R' where
//     R'[l][n] = sum_l' S^-1[l'][l] * Rows[l'][n]          (p x ld, once per walker and window)
// so the flush needs no p x p product per row block.  One warp handles the 8-column tiles
// warp, warp + nwarps, ...: source row l' is src + rowoff_s[l'], the result goes to dst[l * ld + n]
// for l < p.  src (double, or float rows of an fp32-stored inverse) may alias dst (a tile is read
// completely before it is written).
// sinv_s: S^-1 in shared memory, row stride gs.
template <int KMAX, typename TS>
__device__ __forceinline__ void rprime_warp(const double *sinv_s, int gs, int p, const TS *src,
                                            const long long *rowoff_s, double *dst, int ld, int warp,
                                            int nwarps, int lane)
{
    constexpr int MB = KMAX / 8, KQ = KMAX / 4;
    const int g = lane >> 2, t = lane & 3;
    double a[MB][KQ];
    long long off[KQ];
#pragma unroll
    for (int kq = 0; kq < KQ; ++kq) {
        const int lp = 4 * kq + t;
        off[kq] = lp < p ? rowoff_s[lp] : -1;
#pragma unroll
        for (int mb = 0; mb < MB; ++mb) {
            const int l = 8 * mb + g;
            a[mb][kq] = (l < p && lp < p) ? sinv_s[lp * gs + l] : 0.0;
        }
    }
    for (int n0 = 8 * warp; n0 < ld; n0 += 8 * nwarps) {
        double b[KQ], c[MB][2];
#pragma unroll
        for (int kq = 0; kq < KQ; ++kq) b[kq] = off[kq] >= 0 ? (double)src[off[kq] + n0 + g] : 0.0;
#pragma unroll
        for (int mb = 0; mb < MB; ++mb) c[mb][0] = c[mb][1] = 0.0;
#pragma unroll
        for (int kq = 0; kq < KQ; ++kq)
            if (4 * kq < p) {
#pragma unroll
                for (int mb = 0; mb < MB; ++mb)
                    if (8 * mb < p) dmma884(c[mb][0], c[mb][1], a[mb][kq], b[kq]);
            }
#pragma unroll
        for (int mb = 0; mb < MB; ++mb) {
            const int l = 8 * mb + g;
            if (l < p) *reinterpret_cast<double2 *>(dst + (size_t)l * ld + n0 + 2 * t) = make_double2(c[mb][0], c[mb][1]);
        }
    }
}

}  // namespace qmc
