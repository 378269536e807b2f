// Device side of the SPO-VGL gather: stencil weights and the 64-row gather.
// Shared by the standalone qmc_spo_vgl kernel and the batched gather of qmc_sweep (sweep.cu).
#pragma once
#include "common.cuh"

namespace qmc {

// Shared-memory staging of one position's stencil: 64 rows, each with its table offset and
// five Cartesian weights (value, d/dx, d/dy, d/dz, Laplacian).
struct StencilSmem {
    float4 wvg[64];                 // (w_v, w_gx, w_gy, w_gz)
    float wlap[64];
    unsigned long long off[64];     // element offset of row (a,b,c) in the table
    double b1d[3][3][4];            // [dim][deriv order][a]: 1-D weights in fp64
    int cell[3];
};

// 1-D uniform cubic B-spline weights of control points i..i+3 at fraction t (R:A1, R:A2).
__device__ __forceinline__ void bspline1d(double t, double *b, double *db, double *d2b)
{
    const double t2 = t * t, t3 = t2 * t, o = 1.0 - t;
    b[0] = o * o * o * (1.0 / 6.0);
    b[1] = (3.0 * t3 - 6.0 * t2 + 4.0) * (1.0 / 6.0);
    b[2] = (-3.0 * t3 + 3.0 * t2 + 3.0 * t + 1.0) * (1.0 / 6.0);
    b[3] = t3 * (1.0 / 6.0);
    db[0] = -0.5 * o * o;
    db[1] = 0.5 * (3.0 * t2 - 4.0 * t);
    db[2] = 0.5 * (-3.0 * t2 + 2.0 * t + 1.0);
    db[3] = 0.5 * t2;
    d2b[0] = o;
    d2b[1] = 3.0 * t - 2.0;
    d2b[2] = -3.0 * t + 1.0;
    d2b[3] = t;
}

// Fill `st` for Cartesian position r (S1 of the hot path).  All threads of the block call it;
// ends with a __syncthreads().  Index and fraction in fp64 (a 128-point grid needs more than
// fp32 to keep the value within 2e-6), weights rounded to fp32 once.
__device__ __forceinline__ void stage_stencil(const SplineView &sp, double rx, double ry, double rz,
                                              StencilSmem &st)
{
    const int tid = threadIdx.x;
    if (tid < 3) {
        const int d = tid;
        const int n = d == 0 ? sp.nx : (d == 1 ? sp.ny : sp.nz);
        double u = rx * sp.linv[0 + d] + ry * sp.linv[3 + d] + rz * sp.linv[6 + d];
        const double u0 = u;
        u -= floor(u);
        const double s = u * (double)n;
        const double fl = floor(s);
        int i = (int)fl;
        const double t = s - fl;
        bool up = false;
        if (i >= n) { i = 0; up = true; }
        st.cell[d] = i;
        bspline1d(t, st.b1d[d][0], st.b1d[d][1], st.b1d[d][2]);
        if (sp.half_twist[d]) {
            // Half twist along cell vector d (eq. 43, twist angle pi; R:A23): the table is one
            // cell of an antiperiodic function.  Control point i + a lives in image m + (i + a) / n of
            // the cell, m the image of the point itself (one further when u rounded up to 1.0); an odd
            // image flips the sign of that control point's 1-D weights, so the 64 products carry it.
            const double m = floor(u0) + (up ? 1.0 : 0.0);
            const int odd = (int)(m - 2.0 * floor(0.5 * m));
#pragma unroll
            for (int a = 0; a < 4; ++a)
                if ((odd + (i + a) / n) & 1) {
                    st.b1d[d][0][a] = -st.b1d[d][0][a];
                    st.b1d[d][1][a] = -st.b1d[d][1][a];
                    st.b1d[d][2][a] = -st.b1d[d][2][a];
                }
        }
    }
    __syncthreads();
    for (int e = tid; e < 64; e += blockDim.x) {
        const int a = e >> 4, b = (e >> 2) & 3, c = e & 3;
        const double bx = st.b1d[0][0][a], by = st.b1d[1][0][b], bz = st.b1d[2][0][c];
        const double dx = st.b1d[0][1][a], dy = st.b1d[1][1][b], dz = st.b1d[2][1][c];
        const double ex = st.b1d[0][2][a], ey = st.b1d[1][2][b], ez = st.b1d[2][2][c];
        const double w = bx * by * bz;
        const double wx = dx * by * bz, wy = bx * dy * bz, wz = bx * by * dz;
        const double wxx = ex * by * bz, wyy = bx * ey * bz, wzz = bx * by * ez;
        const double wxy = dx * dy * bz, wxz = dx * by * dz, wyz = bx * dy * dz;
        float4 o;
        o.x = (float)w;
        o.y = (float)(sp.jac[0] * wx + sp.jac[1] * wy + sp.jac[2] * wz);
        o.z = (float)(sp.jac[3] * wx + sp.jac[4] * wy + sp.jac[5] * wz);
        o.w = (float)(sp.jac[6] * wx + sp.jac[7] * wy + sp.jac[8] * wz);
        st.wvg[e] = o;
        st.wlap[e] = (float)(sp.metric[0] * wxx + sp.metric[1] * wyy + sp.metric[2] * wzz +
                             2.0 * (sp.metric[3] * wxy + sp.metric[4] * wxz + sp.metric[5] * wyz));
        int ix = st.cell[0] + a, iy = st.cell[1] + b, iz = st.cell[2] + c;
        if (ix >= sp.nx) ix -= sp.nx;
        if (iy >= sp.ny) iy -= sp.ny;
        if (iz >= sp.nz) iz -= sp.nz;
        // grids smaller than 4 points wrap more than once
        ix %= sp.nx; iy %= sp.ny; iz %= sp.nz;
        st.off[e] = (((unsigned long long)ix * sp.ny + iy) * sp.nz + iz) * (unsigned long long)sp.np;
    }
    __syncthreads();
}

// Gather 64 rows for the four orbitals starting at column `col` (multiple of 4, < np).
// Fixed summation order e = 0..63 -> bit-reproducible (R:A11).
template <bool WITH_GL>
__device__ __forceinline__ void gather4(const SplineView &sp, const StencilSmem &st, int col,
                                        float4 &v, float4 &gx, float4 &gy, float4 &gz, float4 &lp)
{
    v = gx = gy = gz = lp = make_float4(0.f, 0.f, 0.f, 0.f);
    const float *base = sp.coefs + col;
#pragma unroll 16
    for (int e = 0; e < 64; ++e) {
        const float4 c = ldg_stream(reinterpret_cast<const float4 *>(base + st.off[e]));
        const float4 w = st.wvg[e];
        v.x = fmaf(w.x, c.x, v.x); v.y = fmaf(w.x, c.y, v.y);
        v.z = fmaf(w.x, c.z, v.z); v.w = fmaf(w.x, c.w, v.w);
        if (WITH_GL) {
            const float wl = st.wlap[e];
            gx.x = fmaf(w.y, c.x, gx.x); gx.y = fmaf(w.y, c.y, gx.y);
            gx.z = fmaf(w.y, c.z, gx.z); gx.w = fmaf(w.y, c.w, gx.w);
            gy.x = fmaf(w.z, c.x, gy.x); gy.y = fmaf(w.z, c.y, gy.y);
            gy.z = fmaf(w.z, c.z, gy.z); gy.w = fmaf(w.z, c.w, gy.w);
            gz.x = fmaf(w.w, c.x, gz.x); gz.y = fmaf(w.w, c.y, gz.y);
            gz.z = fmaf(w.w, c.z, gz.z); gz.w = fmaf(w.w, c.w, gz.w);
            lp.x = fmaf(wl, c.x, lp.x); lp.y = fmaf(wl, c.y, lp.y);
            lp.z = fmaf(wl, c.z, lp.z); lp.w = fmaf(wl, c.w, lp.w);
        }
    }
}

}  // namespace qmc
