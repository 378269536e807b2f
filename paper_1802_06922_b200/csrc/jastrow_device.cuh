// One- and two-body B-spline Jastrow factor (sec 7, eq. 28-33): device-side evaluation shared
// by jastrow.cu (ratio of a single-electron move, value) and window.cu (moves inside a delayed window).
//
//   u(r) = sum_m p_m B_3(r / delta - m),  delta = r_c / M,  B_3 supported on [-3, 1)      (eq. 33)
// For r / delta = i + t, t in [0, 1), only m = i .. i + 3 contribute, with the four weights of the
// uniform cubic B-spline at t -- the same control-point convention as the orbital table (R:A2), here in
// fp64.  Control points beyond p_M do not exist (the sum of eq. 33 stops at M): the table stores three
// zeros behind every function.  u = 0 for r >= r_c (R:A21).
#pragma once
#include "common.cuh"

namespace qmc {

constexpr int kJasMaxFunc = 8;
constexpr int kJasMaxCoef = 256;      // control points of all functions together, padding included

struct JasTable {
    int nfunc;
    int f_same, f_opp;                // electron-electron functions (-1: none)
    int periodic;                     // 0: open boundary conditions
    int ortho;                        // periodic with an orthorhombic cell: one image suffices
    double rc[kJasMaxFunc];
    double dinv[kJasMaxFunc];         // M / r_c
    int off[kJasMaxFunc];             // first control point of function f in p[]
    double p[kJasMaxCoef];
    double lat[9], linv[9];           // rows = cell vectors; u_d = sum_j r_j linv[3 j + d]
};

// eq. 33 in its four-term form.
__device__ __forceinline__ double jas_u(const JasTable &T, int f, double r)
{
    if (f < 0 || !(r < T.rc[f])) return r != r ? r : 0.0;      // beyond the cutoff; NaN in, NaN out
    const double x = r * T.dinv[f];
    const int i = (int)x;
    const double t = x - (double)i, o = 1.0 - t, t2 = t * t, t3 = t2 * t;
    const double *p = T.p + T.off[f] + i;
    const double b0 = o * o * o, b1 = 3.0 * t3 - 6.0 * t2 + 4.0, b2 = -3.0 * t3 + 3.0 * t2 + 3.0 * t + 1.0;
    return (p[0] * b0 + p[1] * b1 + p[2] * b2 + p[3] * t3) * (1.0 / 6.0);
}

// Distance of a and b through the nearest periodic image (the cutoffs are smaller than the
// Wigner-Seitz radius, so at most one image of a pair lies inside any cutoff, and it is the nearest one).
// Orthorhombic cells: rounding the reduced coordinates finds it.  General cells: the 27 neighbours of the
// rounded image are searched.
__device__ __forceinline__ double jas_dist(const JasTable &T, const double a[3], const double b[3])
{
    double d[3] = {a[0] - b[0], a[1] - b[1], a[2] - b[2]};
    if (!T.periodic) return sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double u[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        u[c] = d[0] * T.linv[c] + d[1] * T.linv[3 + c] + d[2] * T.linv[6 + c];
        u[c] -= rint(u[c]);
    }
    if (T.ortho) {
        const double x = u[0] * T.lat[0], y = u[1] * T.lat[4], z = u[2] * T.lat[8];
        return sqrt(x * x + y * y + z * z);
    }
    double best = INFINITY;
    for (int i = -1; i <= 1; ++i)
        for (int j = -1; j <= 1; ++j)
            for (int k = -1; k <= 1; ++k) {
                const double v0 = u[0] + i, v1 = u[1] + j, v2 = u[2] + k;
                const double x = v0 * T.lat[0] + v1 * T.lat[3] + v2 * T.lat[6];
                const double y = v0 * T.lat[1] + v1 * T.lat[4] + v2 * T.lat[7];
                const double z = v0 * T.lat[2] + v1 * T.lat[5] + v2 * T.lat[8];
                const double r2 = x * x + y * y + z * z;
                if (r2 < best || r2 != r2) best = r2;
            }
    return sqrt(best);
}

// u_f(|rnew - c|) - u_f(|rold - c|): what one fixed particle at c contributes to dJ of a move rold -> rnew.
__device__ __forceinline__ double jas_pair_delta(const JasTable &T, int f, const double rnew[3], const double rold[3],
                                                 const double c[3])
{
    return jas_u(T, f, jas_dist(T, rnew, c)) - jas_u(T, f, jas_dist(T, rold, c));
}

}  // namespace qmc

// The Jastrow handle: the function table and the ions, on the device.
struct qmc_jastrow {
    qmc::JasTable host;       // host copy (shape checks)
    qmc::JasTable *table;     // device
    int nion;
    double *ion;              // device [nion][3]
    int *ion_func;            // device [nion]
    int device;
};
