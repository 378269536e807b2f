/*
 * qmc_oracle.c -- TEST INFRASTRUCTURE.  Plain, slow, fp64 CPU oracle for the
 * particle-by-particle move of arxiv 1802.06922 (QMCPACK overview paper).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares no code, header,
 * table or helper with the CUDA path under paper_1802_06922_b200/csrc/.
 *
 * What it computes, and the passage each function follows (PAPER.md line /
 * section; "R:Ax" = a reading listed in DESIGN.md section 3 where the paper is
 * silent):
 *
 *   orc_spline_vgl    PAPER.md L307-311 (sec 6.2.1): orbitals in "a regular 3D
 *                     B-spline representation", "a constant 64 coefficients ...
 *                     to evaluate each single-particle wavefunction", periodic
 *                     boundary conditions (L307).  Basis = uniform cardinal
 *                     cubic B-spline (R:A1); control points i..i+3, the support
 *                     convention of eq. 33, L369-373 (R:A2); Cartesian gradient
 *                     and Laplacian (R:A6), needed by eq. 3 / eq. 13.
 *   orc_lu_inverse    L325: Slater matrix M_ij = phi_j(r_i); its inverse,
 *                     log|det| and sign by plain LU with partial pivoting.
 *   orc_det_ratio     L299 "for single electron moves": det A'/det A when row k
 *                     of A is replaced by phi(r') = sum_j phi_j(r') Ainv[j][k].
 *   orc_sm_update     L299 "the Sherman-Morrison algorithm, as described in
 *                     [49]": the rank-1 row-replacement update of the inverse.
 *   orc_sweep         L195-199 (sec 5.2.1): "particle-by-particle moves work by
 *                     iterating sequentially over all electrons"; proposal
 *                     eq. 13 with F = 0; acceptance eq. 12 with symmetric T and
 *                     a determinant-only Psi: accept iff R*R > u (R:A8).
 *
 *   orc_sweep_ex      the same with options: (i) drift moves, L183-199: the proposal of eq. 13 with
 *                     the wavefunction force F = 2 grad log Psi_T (L156) and the acceptance of
 *                     eq. 12 with the ratio T(r'->r)/T(r->r') of the Gaussians of eq. 11 / eq. 13
 *                     (R:A20: lambda = 1/2); (ii) single-precision storage of the inverse, L82
 *                     "single, double and mixed precision" (R:A19: B rounded to fp32 when stored,
 *                     all arithmetic in fp64), with orc_init_walkers as the recompute-from-scratch.
 *
 *   orc_spline_vgl_twist   L449-455 (sec 9.2, eq. 43): the same evaluation for real orbitals at a
 *                     half twist, twist angle pi along chosen cell vectors (R:A23): the table is
 *                     one cell of an antiperiodic function.  Pins: tests/test_twist_pins.py.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): partition of unity,
 * polynomial reproduction, plane-wave node closed form, periodicity, C2
 * continuity, scipy.interpolate.BSpline tensor product, central finite
 * differences, Leibniz / numpy determinants (N <= 16), numpy inverse,
 * log-det telescoping, accept control flow.  Every function here is pinned.
 *
 * Layouts (all row-major, caller-owned):
 *   lattice[9]   rows = cell vectors a0,a1,a2;  r = u . lattice
 *   coefs        float [nx][ny][nz][norb], periodic, no halo (R:A3, R:A4)
 *   pos          double [..][3] Cartesian
 *   B            double [n][n] = (A^-1)^T, so row k of B is column k of A^-1,
 *                "the moved electron's inverse-matrix row"
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------- */
/* 3x3 inverse: Li = L^-1.  Returns 0 on success, -1 if singular.            */
static int inv3(const double L[9], double Li[9])
{
    double c00 = L[4] * L[8] - L[5] * L[7];
    double c01 = L[5] * L[6] - L[3] * L[8];
    double c02 = L[3] * L[7] - L[4] * L[6];
    double det = L[0] * c00 + L[1] * c01 + L[2] * c02;
    if (det == 0.0 || !isfinite(det)) return -1;
    Li[0] = c00 / det;
    Li[1] = (L[2] * L[7] - L[1] * L[8]) / det;
    Li[2] = (L[1] * L[5] - L[2] * L[4]) / det;
    Li[3] = c01 / det;
    Li[4] = (L[0] * L[8] - L[2] * L[6]) / det;
    Li[5] = (L[2] * L[3] - L[0] * L[5]) / det;
    Li[6] = c02 / det;
    Li[7] = (L[1] * L[6] - L[0] * L[7]) / det;
    Li[8] = (L[0] * L[4] - L[1] * L[3]) / det;
    return 0;
}

/* Uniform cubic B-spline weights of the four control points i..i+3 at
 * fractional offset t in [0,1), with first and second derivatives in t. */
static void bspline_weights(double t, double b[4], double db[4], double d2b[4])
{
    double t2 = t * t, t3 = t2 * t, o = 1.0 - t;
    b[0] = o * o * o / 6.0;
    b[1] = (3.0 * t3 - 6.0 * t2 + 4.0) / 6.0;
    b[2] = (-3.0 * t3 + 3.0 * t2 + 3.0 * t + 1.0) / 6.0;
    b[3] = t3 / 6.0;
    db[0] = -o * o / 2.0;
    db[1] = (3.0 * t2 - 4.0 * t) / 2.0;
    db[2] = (-3.0 * t2 + 2.0 * t + 1.0) / 2.0;
    db[3] = t2 / 2.0;
    d2b[0] = o;
    d2b[1] = 3.0 * t - 2.0;
    d2b[2] = -3.0 * t + 1.0;
    d2b[3] = t;
}

/* Reduced coordinate -> (cell index, fraction) along one dimension (R:A7). */
static void cell_of(double u, int n, int *i, double *t)
{
    if (!isfinite(u)) { *i = 0; *t = u - u; return; } /* NaN weights: every orbital is NaN (R:A18) */
    u -= floor(u);
    double s = u * (double)n;
    double fl = floor(s);
    int ii = (int)fl;
    *t = s - fl;
    if (ii >= n) ii = 0; /* u rounded up to 1.0: same point as u = 0 */
    *i = ii;
}

/*
 * Value, Cartesian gradient and Laplacian of all norb orbitals at npos
 * positions.  v [npos][norb], g [npos][3][norb], l [npos][norb], all double;
 * g and l may be NULL.  Returns 0, or -1 on bad arguments.
 */
static int spline_vgl_tw(int nx, int ny, int nz, int norb, const double lattice[9],
                         const float *coefs, int npos, const double *pos, const int *half_twist,
                         double *v, double *g, double *l)
{
    double Li[9];
    if (nx < 1 || ny < 1 || nz < 1 || norb < 1 || npos < 0) return -1;
    if (inv3(lattice, Li) != 0) return -1;
    const int nd[3] = {nx, ny, nz};
    /* J[j][d] = d s_d / d r_j = Li[j][d] * N_d */
    double J[3][3];
    for (int j = 0; j < 3; ++j)
        for (int d = 0; d < 3; ++d) J[j][d] = Li[3 * j + d] * (double)nd[d];

    double *acc = (double *)malloc((size_t)norb * 10 * sizeof(double));
    if (!acc) return -1;
    double *a_v = acc, *a_d = acc + norb, *a_h = acc + 4 * (size_t)norb;

    for (int p = 0; p < npos; ++p) {
        const double *r = pos + 3 * (size_t)p;
        int i[3];
        double t[3], b[3][4], db[3][4], d2b[3][4];
        for (int d = 0; d < 3; ++d) {
            double u = r[0] * Li[0 + d] + r[1] * Li[3 + d] + r[2] * Li[6 + d];
            cell_of(u, nd[d], &i[d], &t[d]);
            bspline_weights(t[d], b[d], db[d], d2b[d]);
            if (half_twist && half_twist[d] && isfinite(u)) {
                /* Twist angle pi along cell vector d (eq. 43 with Theta_d = pi; R:A23):
                 * the table holds one cell of an ANTIPERIODIC function, c[i + m n] = (-1)^m c[i].
                 * The point lies in image floor(u) (one more when u - floor(u) rounded up to 1.0
                 * and cell_of moved it to u = 0, R:A7); control point i + a lies (i + a) / n
                 * images further on. */
                double fu = floor(u);
                long long img = (long long)fmod(fu, 2.0);
                if ((u - fu) * (double)nd[d] >= (double)nd[d]) img += 1;
                for (int a = 0; a < 4; ++a)
                    if ((img + (i[d] + a) / nd[d]) & 1) {
                        b[d][a] = -b[d][a];
                        db[d][a] = -db[d][a];
                        d2b[d][a] = -d2b[d][a];
                    }
            }
        }
        memset(acc, 0, (size_t)norb * 10 * sizeof(double));
        for (int a = 0; a < 4; ++a)
            for (int bb = 0; bb < 4; ++bb)
                for (int c = 0; c < 4; ++c) {
                    size_t ix = (size_t)((i[0] + a) % nx);
                    size_t iy = (size_t)((i[1] + bb) % ny);
                    size_t iz = (size_t)((i[2] + c) % nz);
                    const float *row = coefs + ((ix * ny + iy) * nz + iz) * (size_t)norb;
                    double w = b[0][a] * b[1][bb] * b[2][c];
                    double wx = db[0][a] * b[1][bb] * b[2][c];
                    double wy = b[0][a] * db[1][bb] * b[2][c];
                    double wz = b[0][a] * b[1][bb] * db[2][c];
                    double wxx = d2b[0][a] * b[1][bb] * b[2][c];
                    double wyy = b[0][a] * d2b[1][bb] * b[2][c];
                    double wzz = b[0][a] * b[1][bb] * d2b[2][c];
                    double wxy = db[0][a] * db[1][bb] * b[2][c];
                    double wxz = db[0][a] * b[1][bb] * db[2][c];
                    double wyz = b[0][a] * db[1][bb] * db[2][c];
                    for (int n = 0; n < norb; ++n) {
                        double cf = (double)row[n];
                        a_v[n] += w * cf;
                        a_d[0 * (size_t)norb + n] += wx * cf;
                        a_d[1 * (size_t)norb + n] += wy * cf;
                        a_d[2 * (size_t)norb + n] += wz * cf;
                        a_h[0 * (size_t)norb + n] += wxx * cf;
                        a_h[1 * (size_t)norb + n] += wyy * cf;
                        a_h[2 * (size_t)norb + n] += wzz * cf;
                        a_h[3 * (size_t)norb + n] += wxy * cf;
                        a_h[4 * (size_t)norb + n] += wxz * cf;
                        a_h[5 * (size_t)norb + n] += wyz * cf;
                    }
                }
        for (int n = 0; n < norb; ++n) {
            v[(size_t)p * norb + n] = a_v[n];
            double d1[3] = {a_d[n], a_d[(size_t)norb + n], a_d[2 * (size_t)norb + n]};
            /* symmetric Hessian in grid coordinates s */
            double h[3][3];
            h[0][0] = a_h[0 * (size_t)norb + n];
            h[1][1] = a_h[1 * (size_t)norb + n];
            h[2][2] = a_h[2 * (size_t)norb + n];
            h[0][1] = h[1][0] = a_h[3 * (size_t)norb + n];
            h[0][2] = h[2][0] = a_h[4 * (size_t)norb + n];
            h[1][2] = h[2][1] = a_h[5 * (size_t)norb + n];
            if (g)
                for (int j = 0; j < 3; ++j)
                    g[((size_t)p * 3 + j) * norb + n] =
                        J[j][0] * d1[0] + J[j][1] * d1[1] + J[j][2] * d1[2];
            if (l) {
                double lap = 0.0;
                for (int j = 0; j < 3; ++j)
                    for (int d = 0; d < 3; ++d)
                        for (int e = 0; e < 3; ++e) lap += J[j][d] * J[j][e] * h[d][e];
                l[(size_t)p * norb + n] = lap;
            }
        }
    }
    free(acc);
    return 0;
}

int orc_spline_vgl(int nx, int ny, int nz, int norb, const double lattice[9],
                   const float *coefs, int npos, const double *pos,
                   double *v, double *g, double *l)
{
    return spline_vgl_tw(nx, ny, nz, norb, lattice, coefs, npos, pos, NULL, v, g, l);
}

/*
 * The same evaluation for real orbitals at a half twist (sec 9.2, eq. 43 with
 * twist angle Theta_d = pi along every cell vector d with half_twist[d] != 0, 0 along the others):
 * phi(r + L_d) = -phi(r).  half_twist = {0,0,0} is orc_spline_vgl.  Reading R:A23 in DESIGN.md.
 */
int orc_spline_vgl_twist(int nx, int ny, int nz, int norb, const double lattice[9],
                         const float *coefs, int npos, const double *pos, const int half_twist[3],
                         double *v, double *g, double *l)
{
    if (!half_twist) return -1;
    return spline_vgl_tw(nx, ny, nz, norb, lattice, coefs, npos, pos, half_twist, v, g, l);
}

/* ------------------------------------------------------------------------- */
/*
 * Plain LU with partial pivoting of the n x n matrix A (row-major, not
 * modified).  Writes Ainv (row-major, n x n; may be NULL), log|det A| and the
 * sign of det A.  Returns 0, -4 if a pivot is exactly zero (singular), -2 on
 * allocation failure.
 */
int orc_lu_inverse(int n, const double *A, double *Ainv, double *logdet, int *sign)
{
    size_t nn = (size_t)n * n;
    double *LU = (double *)malloc(nn * sizeof(double));
    int *piv = (int *)malloc((size_t)n * sizeof(int));
    double *col = (double *)malloc((size_t)n * sizeof(double));
    if (!LU || !piv || !col) { free(LU); free(piv); free(col); return -2; }
    memcpy(LU, A, nn * sizeof(double));
    double ld = 0.0;
    int sg = 1, rc = 0;
    for (int k = 0; k < n; ++k) {
        int p = k;
        double best = fabs(LU[(size_t)k * n + k]);
        for (int i = k + 1; i < n; ++i) {
            double x = fabs(LU[(size_t)i * n + k]);
            if (x > best) { best = x; p = i; }
        }
        piv[k] = p;
        if (p != k) {
            for (int j = 0; j < n; ++j) {
                double tmp = LU[(size_t)k * n + j];
                LU[(size_t)k * n + j] = LU[(size_t)p * n + j];
                LU[(size_t)p * n + j] = tmp;
            }
            sg = -sg;
        }
        double d = LU[(size_t)k * n + k];
        if (d == 0.0 || !isfinite(d)) { rc = -4; break; }
        ld += log(fabs(d));
        if (d < 0.0) sg = -sg;
        for (int i = k + 1; i < n; ++i) {
            double f = LU[(size_t)i * n + k] / d;
            LU[(size_t)i * n + k] = f;
            for (int j = k + 1; j < n; ++j) LU[(size_t)i * n + j] -= f * LU[(size_t)k * n + j];
        }
    }
    if (rc == 0) {
        if (logdet) *logdet = ld;
        if (sign) *sign = sg;
        if (Ainv) {
            /* solve A x = e_c for every unit vector e_c */
            for (int c = 0; c < n; ++c) {
                for (int i = 0; i < n; ++i) col[i] = (i == c) ? 1.0 : 0.0;
                for (int k = 0; k < n; ++k) {
                    int p = piv[k];
                    if (p != k) { double tmp = col[k]; col[k] = col[p]; col[p] = tmp; }
                }
                for (int i = 0; i < n; ++i) {
                    double s = col[i];
                    for (int j = 0; j < i; ++j) s -= LU[(size_t)i * n + j] * col[j];
                    col[i] = s;
                }
                for (int i = n - 1; i >= 0; --i) {
                    double s = col[i];
                    for (int j = i + 1; j < n; ++j) s -= LU[(size_t)i * n + j] * col[j];
                    col[i] = s / LU[(size_t)i * n + i];
                }
                for (int i = 0; i < n; ++i) Ainv[(size_t)i * n + c] = col[i];
            }
        }
    }
    free(LU); free(piv); free(col);
    return rc;
}

/* B = (A^-1)^T from A, with log|det A| and sign.  Same return codes. */
int orc_binv_from_A(int n, const double *A, double *B, double *logdet, int *sign)
{
    size_t nn = (size_t)n * n;
    double *Ai = (double *)malloc(nn * sizeof(double));
    if (!Ai) return -2;
    int rc = orc_lu_inverse(n, A, Ai, logdet, sign);
    if (rc == 0)
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j) B[(size_t)i * n + j] = Ai[(size_t)j * n + i];
    free(Ai);
    return rc;
}

/* R = sum_j phi[j] * Ainv[j][k] = sum_j B[k][j] * phi[j]   (L299) */
double orc_det_ratio(int n, const double *B, int k, const double *phi)
{
    double r = 0.0;
    for (int j = 0; j < n; ++j) r += B[(size_t)k * n + j] * phi[j];
    return r;
}

/*
 * Sherman-Morrison update of B = (A^-1)^T when row k of A is replaced by phi,
 * R = orc_det_ratio(n, B, k, phi):
 *     w_m = sum_j B[m][j] phi[j]
 *     B'[m][j] = B[m][j] - (w_m - delta_mk) * B[k][j] / R
 */
int orc_sm_update(int n, double *B, int k, const double *phi, double R)
{
    double *w = (double *)malloc((size_t)n * sizeof(double));
    double *rowk = (double *)malloc((size_t)n * sizeof(double));
    if (!w || !rowk) { free(w); free(rowk); return -2; }
    for (int m = 0; m < n; ++m) {
        double s = 0.0;
        for (int j = 0; j < n; ++j) s += B[(size_t)m * n + j] * phi[j];
        w[m] = s;
    }
    memcpy(rowk, B + (size_t)k * n, (size_t)n * sizeof(double));
    for (int m = 0; m < n; ++m) {
        double f = (w[m] - (m == k ? 1.0 : 0.0)) / R;
        for (int j = 0; j < n; ++j) B[(size_t)m * n + j] -= f * rowk[j];
    }
    free(w); free(rowk);
    return 0;
}

/* ------------------------------------------------------------------------- */
/*
 * Particle-by-particle sweep (L195-199), walkers independent (L181).
 *
 *   pos     [nw][nel][3]  in/out, stored unwrapped
 *   B       [nw][nel][nel] in/out, (A^-1)^T of the current Slater matrix
 *   A       [nw][nel][nel] in/out or NULL; the Slater matrix itself, row i =
 *           phi(r_i).  Required when mode == 1.
 *   logdet  [nw], sign [nw]  in/out: log|det A|, sign(det A)
 *   delta   [nsweeps][nel][nw][3]  pre-generated Gaussian displacements
 *   unif    [nsweeps][nel][nw]     pre-generated uniforms in [0,1)
 *   iel_count  electrons moved per sweep (0..iel_count-1); nel for a full one
 *   ratios_out / accept_out  [nsweeps][nel][nw] or NULL
 *   forced  NULL, or decisions to impose instead of the Metropolis test
 *   phi_in  NULL, or float [nsweeps][nel][nw][nel]: orbital vectors to use
 *           instead of evaluating the spline ("identical orbital vectors")
 *   phi_out NULL, or double [nsweeps][nel][nw][nel]: the vectors used
 *   mode    0 = Sherman-Morrison update on accept (orc_sm_update);
 *           1 = definitional: recompute B by LU from A after every accept
 *   bnorm_out  NULL, or [nsweeps][nel][nw]: sum_j |B[k][j]| of the row used by each ratio (a
 *           diagnostic: it bounds how an error in phi propagates into R)
 *   nthreads  OpenMP threads over walkers (<=1: serial)
 *   fixed_node  != 0: the fixed-node rule of PAPER.md L253 -- "proposed moves that result in a
 *           nodal crossing are detected through the change in sign of the wavefunction and are
 *           rejected": a move with R < 0 is rejected whatever u is (ignored when `forced`)
 *   force_out  NULL, or double [nsweeps][nel][nw][3]: the "wavefunction force" F = 2 grad log Psi_T
 *           (the F of eq. 11 / eq. 13) on the moved electron at the PROPOSED
 *           configuration.  With Psi = det A, row k replaced by phi(r'):
 *               grad_k log|det A'| = sum_j grad phi_j(r') (A'^-1)[j][k]
 *                                  = sum_j grad phi_j(r') B[k][j] / R        (B'[k] = B[k] / R)
 *           The gradients come from this oracle's own fp64 spline at r' (also in phi_in mode).
 *           Written for every move, accepted or not; 0 when R == 0.
 *
 * Accept iff R*R > u; a non-finite R is rejected (R:A8); an imposed accept (`forced`) of a move
 * whose R is zero or not finite is refused -- the update divides by R and the new Slater matrix
 * would be singular (R:A18).  On accept:
 * r_k <- r_k + delta (one fp64 add), row k of A <- phi, log|det| += log|R|,
 * sign *= sgn(R), B updated.  Returns 0 or the first error code met.
 */
/*
 * Options of orc_sweep_ex (all zero / NULL = orc_sweep).
 *
 * Drift moves (R:A20).  tau > 0 switches them on.  With lambda = 1/2 (electrons,
 * Hartree atomic units) eq. 13 reads T(r_k -> r_k') ~ exp(-|r_k' - r_k - tau F_k(r)|^2 / (2 tau)),
 * i.e. r_k' = r_k + tau F_k(r) + chi with chi ~ N(0, tau) per component (eq. 19 for one electron);
 * `delta` holds chi.  F_k(r) = 2 grad_k log|det A| = 2 sum_j grad phi_j(r_k) B[k][j] at the CURRENT
 * configuration (L156); F_k(r') = 2 sum_j grad phi_j(r_k') B[k][j] / R at the proposed one.  The
 * move is accepted with the probability of eq. 12,
 *     min(1, R^2 T(r'->r) / T(r->r')),   log T(r'->r)/T(r->r') = (|chi|^2 - |r_k - r_k' - tau F_k(r')|^2) / (2 tau),
 * i.e. iff R^2 exp(logT) > u.  With tau -> 0+ ... the no-drift walk is NOT recovered by tau = 0 (that
 * switches drift off and uses delta as the whole displacement, eq. 13 with F = 0).
 *   rprop_in   NULL, or [nsweeps][nel][nw][3]: proposed positions to use instead of r + tau F + chi
 *              (replay of another implementation's proposals; the forward density still uses this
 *              oracle's own F_k(r): log T = (|r_k' - r_k - tau F_k(r)|^2 - |r_k - r_k' - tau F_k(r')|^2) / (2 tau))
 *   rprop_out  NULL, or same shape: the proposed positions used
 *   fcur_out   NULL, or [nsweeps][nel][nw][3]: F_k(r) at the current configuration
 *   logt_out   NULL, or [nsweeps][nel][nw]: log T(r'->r)/T(r->r')  (-inf... finite only when R != 0)
 *
 * Single-precision storage of the inverse (R:A19).  b32 != 0: B holds values that are
 * exactly representable in fp32 on entry (the caller rounds the initial inverse) and is rounded to
 * fp32 (round to nearest even, the C cast) whenever it is STORED: after every accepted update when
 * b32 == 1 (rank-1 Sherman-Morrison), or -- b32 = K >= 2, the delayed update of rank K -- when a
 * window of K consecutive electron steps closes (k % K == K - 1 within the moved range, or the end of
 * the sweep), the accepted updates inside the window being applied in fp64 to the unrounded matrix.
 * Ratios, Sherman-Morrison multipliers and log|det| are fp64 arithmetic on those stored values.
 */
typedef struct orc_sweep_opts {
    double tau;
    const double *rprop_in;
    double *rprop_out, *fcur_out, *logt_out;
    int b32;
    /* Jastrow factor (eq. 26, eq. 28-33; qmc_jastrow_oracle.c): Psi_T = e^{-J} D, so the move of
     * electron k has |Psi'/Psi|^2 = R^2 exp(-2 dJ), dJ = orc_jastrow_dj at the walker's CURRENT positions;
     * the move is accepted iff R^2 exp(-2 dJ) > u (eq. 12, symmetric T).  `other` holds the electrons of the
     * other spin, [nw][nother][3], fixed during this sweep.  Not combined with drift moves (the drift
     * would need grad J, which is not built): tau > 0 with a Jastrow factor is an error. */
    const struct orc_jastrow *jas;
    const double *other;
    int nother;
    double *jratio_out;    /* NULL, or [nsweeps][nel][nw]: exp(-dJ) of every move */
} orc_sweep_opts;

struct orc_jastrow;
double orc_jastrow_dj(const struct orc_jastrow *J, int nel, const double *pos, int nother, const double *other,
                      int k, const double rnew[3]);

static void round_to_fp32(double *x, size_t n)
{
    for (size_t i = 0; i < n; ++i) x[i] = (double)(float)x[i];
}

int orc_sweep_ex(int nx, int ny, int nz, int norb, const double lattice[9], const float *coefs,
              int nw, int nel, double *pos, double *B, double *A, double *logdet, int *sign,
              const double *delta, const double *unif, int nsweeps, int iel_count,
              double *ratios_out, unsigned char *accept_out, const unsigned char *forced,
              const float *phi_in, double *phi_out, int mode, int nthreads, double *bnorm_out,
              int fixed_node, double *force_out, const orc_sweep_opts *opts)
{
    if (nel != norb || nw < 0 || nsweeps < 0 || iel_count < 0 || iel_count > nel) return -1;
    if (mode == 1 && !A) return -1;
    const double tau = opts ? opts->tau : 0.0;
    const int drift = tau > 0.0;
    const int b32 = opts ? opts->b32 : 0;
    const double *rprop_in = opts ? opts->rprop_in : NULL;
    double *rprop_out = opts ? opts->rprop_out : NULL;
    double *fcur_out = opts ? opts->fcur_out : NULL;
    double *logt_out = opts ? opts->logt_out : NULL;
    if (b32 < 0 || (opts && opts->tau < 0.0)) return -1;
    const struct orc_jastrow *jas = opts ? opts->jas : NULL;
    if (jas && drift) return -1;
    int rc_all = 0;
    size_t nn = (size_t)nel * nel;
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
    for (int w = 0; w < nw; ++w) {
        double *phi = (double *)malloc((size_t)nel * sizeof(double));
        const int want_grad = force_out || drift;
        double *grad = want_grad ? (double *)malloc((size_t)4 * nel * sizeof(double)) : NULL;   /* 3 gradients + scratch values */
        double *Bw = B + (size_t)w * nn;
        double *Aw = A ? A + (size_t)w * nn : NULL;
        int rc = (phi && (grad || !want_grad)) ? 0 : -2;
        for (int s = 0; s < nsweeps && rc == 0; ++s)
            for (int k = 0; k < iel_count && rc == 0; ++k) {
                size_t mv = ((size_t)s * nel + k) * nw + w;
                double *rk = pos + ((size_t)w * nel + k) * 3;
                double fcur[3] = {0.0, 0.0, 0.0};
                if (drift) {           /* F_k(r) = 2 sum_j grad phi_j(r_k) B[k][j], current configuration */
                    rc = orc_spline_vgl(nx, ny, nz, norb, lattice, coefs, 1, rk, grad + (size_t)3 * nel, grad, NULL);
                    if (rc) break;
                    for (int d = 0; d < 3; ++d) {
                        double gd = 0.0;
                        for (int j = 0; j < nel; ++j) gd += grad[(size_t)d * nel + j] * Bw[(size_t)k * nel + j];
                        fcur[d] = 2.0 * gd;
                    }
                    if (fcur_out) { fcur_out[3 * mv] = fcur[0]; fcur_out[3 * mv + 1] = fcur[1]; fcur_out[3 * mv + 2] = fcur[2]; }
                }
                double rnew[3];
                for (int d = 0; d < 3; ++d) {
                    if (drift && rprop_in) rnew[d] = rprop_in[3 * mv + d];
                    else if (drift) rnew[d] = rk[d] + (tau * fcur[d] + delta[3 * mv + d]);
                    else rnew[d] = rk[d] + delta[3 * mv + d];
                }
                if (rprop_out) { rprop_out[3 * mv] = rnew[0]; rprop_out[3 * mv + 1] = rnew[1]; rprop_out[3 * mv + 2] = rnew[2]; }
                if (phi_in) {
                    for (int j = 0; j < nel; ++j) phi[j] = (double)phi_in[mv * nel + j];
                } else {
                    rc = orc_spline_vgl(nx, ny, nz, norb, lattice, coefs, 1, rnew, phi, NULL, NULL);
                    if (rc) break;
                }
                if (phi_out) memcpy(phi_out + mv * nel, phi, (size_t)nel * sizeof(double));
                double R = orc_det_ratio(nel, Bw, k, phi);
                double fnew[3] = {0.0, 0.0, 0.0}, logt = 0.0;
                if (want_grad) {       /* F = 2 grad_k log|det A'| at the proposed configuration */
                    rc = orc_spline_vgl(nx, ny, nz, norb, lattice, coefs, 1, rnew, grad + (size_t)3 * nel, grad, NULL);
                    if (rc) break;
                    for (int d = 0; d < 3; ++d) {
                        double gd = 0.0;
                        for (int j = 0; j < nel; ++j) gd += grad[(size_t)d * nel + j] * Bw[(size_t)k * nel + j];
                        fnew[d] = (R != 0.0) ? 2.0 * gd / R : 0.0;
                        if (force_out) force_out[3 * mv + d] = fnew[d];
                    }
                }
                if (drift) {           /* log T(r'->r)/T(r->r'), eq. 11-13 with lambda = 1/2 */
                    double fwd = 0.0, bwd = 0.0;
                    for (int d = 0; d < 3; ++d) {
                        double a = rnew[d] - rk[d] - tau * fcur[d];
                        double b = rk[d] - rnew[d] - tau * fnew[d];
                        fwd += a * a;
                        bwd += b * b;
                    }
                    logt = (fwd - bwd) / (2.0 * tau);
                    if (logt_out) logt_out[mv] = logt;
                }
                double jfac2 = 1.0;    /* exp(-2 dJ): the Jastrow part of |Psi'/Psi|^2 */
                if (jas) {
                    double dj = orc_jastrow_dj(jas, nel, pos + (size_t)w * nel * 3, opts->nother,
                                               opts->other ? opts->other + (size_t)w * opts->nother * 3 : NULL, k, rnew);
                    jfac2 = exp(-2.0 * dj);
                    if (opts->jratio_out) opts->jratio_out[mv] = exp(-dj);
                }
                int acc;
                if (forced) acc = forced[mv] != 0 && isfinite(R) && R != 0.0; /* R:A18 */
                else if (jas) acc = isfinite(R) && isfinite(jfac2) && (R * R * jfac2 > unif[mv]) && !(fixed_node && R < 0.0);
                else if (drift) acc = isfinite(R) && isfinite(logt) && (R * R * exp(logt) > unif[mv]) && !(fixed_node && R < 0.0);
                else acc = isfinite(R) && (R * R > unif[mv]) && !(fixed_node && R < 0.0);
                if (ratios_out) ratios_out[mv] = R;
                if (bnorm_out) {
                    double bn = 0.0;
                    for (int j = 0; j < nel; ++j) bn += fabs(Bw[(size_t)k * nel + j]);
                    bnorm_out[mv] = bn;
                }
                if (accept_out) accept_out[mv] = (unsigned char)acc;
                if (acc) {
                    rk[0] = rnew[0]; rk[1] = rnew[1]; rk[2] = rnew[2];
                    if (Aw) memcpy(Aw + (size_t)k * nel, phi, (size_t)nel * sizeof(double));
                    logdet[w] += log(fabs(R));
                    if (R < 0.0) sign[w] = -sign[w];
                    if (mode == 1) rc = orc_binv_from_A(nel, Aw, Bw, NULL, NULL);
                    else rc = orc_sm_update(nel, Bw, k, phi, R);
                    if (b32 == 1) round_to_fp32(Bw, nn);
                }
                /* delayed rank-K storage: the window of K steps closes here (R:A19) */
                if (b32 >= 2 && (k % b32 == b32 - 1 || k == iel_count - 1)) round_to_fp32(Bw, nn);
            }
        free(phi);
        free(grad);
        if (rc) {
#ifdef _OPENMP
#pragma omp critical
#endif
            if (!rc_all) rc_all = rc;
        }
    }
    return rc_all;
}

int orc_sweep(int nx, int ny, int nz, int norb, const double lattice[9], const float *coefs,
              int nw, int nel, double *pos, double *B, double *A, double *logdet, int *sign,
              const double *delta, const double *unif, int nsweeps, int iel_count,
              double *ratios_out, unsigned char *accept_out, const unsigned char *forced,
              const float *phi_in, double *phi_out, int mode, int nthreads, double *bnorm_out,
              int fixed_node, double *force_out)
{
    return orc_sweep_ex(nx, ny, nz, norb, lattice, coefs, nw, nel, pos, B, A, logdet, sign, delta, unif,
                        nsweeps, iel_count, ratios_out, accept_out, forced, phi_in, phi_out, mode, nthreads,
                        bnorm_out, fixed_node, force_out, NULL);
}

/* Slater matrices A[w][i][j] = phi_j(r_{w,i}) (L325) for nw walkers. */
int orc_slater_matrix(int nx, int ny, int nz, int norb, const double lattice[9],
                      const float *coefs, int nw, int nel, const double *pos, double *A)
{
    if (nel != norb) return -1;
    return orc_spline_vgl(nx, ny, nz, norb, lattice, coefs, nw * nel, pos, A, NULL, NULL);
}

/* Slater matrix, B = (A^-1)^T, log|det| and sign of every walker (walkers are independent,
 * L181: OpenMP over walkers).  A may be NULL.  Returns 0 or the first error code met. */
int orc_init_walkers(int nx, int ny, int nz, int norb, const double lattice[9], const float *coefs,
                     int nw, int nel, const double *pos, double *A, double *B, double *logdet,
                     int *sign, int nthreads)
{
    if (nel != norb) return -1;
    int rc_all = 0;
    size_t nn = (size_t)nel * nel;
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic) num_threads(nthreads)
#endif
    for (int w = 0; w < nw; ++w) {
        double *Aw = A ? A + (size_t)w * nn : (double *)malloc(nn * sizeof(double));
        int rc = Aw ? 0 : -2;
        if (!rc) rc = orc_spline_vgl(nx, ny, nz, norb, lattice, coefs, nel, pos + (size_t)w * nel * 3, Aw, NULL, NULL);
        if (!rc) rc = orc_binv_from_A(nel, Aw, B + (size_t)w * nn, logdet + w, sign + w);
        if (!A) free(Aw);
        if (rc) {
#ifdef _OPENMP
#pragma omp critical
#endif
            if (!rc_all) rc_all = rc;
        }
    }
    return rc_all;
}

/* ---------------------------------------------------------------------------
 * orc_det_kinetic -- the determinant's contribution to the kinetic term of the local energy,
 * E_L,kin = Psi^-1 (-1/2 sum_i lap_i) Psi (eq. 3 first term, eq. 37; L401: collected
 * after all walkers have advanced one step).  For Psi = det A, A_ij = phi_j(r_i), only row i of A
 * depends on r_i, so by the cofactor expansion along that row
 *     grad_i det A / det A = sum_j grad phi_j(r_i) (A^-1)[j][i] = sum_j grad phi_j(r_i) B[i][j]
 *     lap_i  det A / det A = sum_j lap  phi_j(r_i) B[i][j]
 * and, as a consistency check of (pos, B), one[w][i] = sum_j phi_j(r_i) B[i][j] = 1.
 *
 *   pos  [nw][nel][3], B [nw][nel][nel] = (A^-1)^T
 *   grad_out [nw][nel][3], lap_out [nw][nel], one_out [nw][nel] (any may be NULL)
 *   ekin_out [nw] = -1/2 sum_i lap_out[w][i]                      (may be NULL)
 */
int orc_det_kinetic(int nx, int ny, int nz, int norb, const double lattice[9], const float *coefs,
                    int nw, int nel, const double *pos, const double *B, double *grad_out,
                    double *lap_out, double *one_out, double *ekin_out)
{
    if (nel != norb || nw < 0) return -1;
    double *v = (double *)malloc((size_t)5 * nel * sizeof(double));
    if (!v) return -2;
    double *g = v + nel, *l = v + (size_t)4 * nel;
    int rc = 0;
    for (int w = 0; w < nw && rc == 0; ++w) {
        double ek = 0.0;
        for (int i = 0; i < nel && rc == 0; ++i) {
            const double *Bi = B + ((size_t)w * nel + i) * nel;
            rc = orc_spline_vgl(nx, ny, nz, norb, lattice, coefs, 1, pos + ((size_t)w * nel + i) * 3, v, g, l);
            if (rc) break;
            double one = 0.0, gx = 0.0, gy = 0.0, gz = 0.0, lp = 0.0;
            for (int j = 0; j < nel; ++j) {
                one += v[j] * Bi[j];
                gx += g[j] * Bi[j];
                gy += g[(size_t)nel + j] * Bi[j];
                gz += g[(size_t)2 * nel + j] * Bi[j];
                lp += l[j] * Bi[j];
            }
            if (grad_out) {
                double *go = grad_out + ((size_t)w * nel + i) * 3;
                go[0] = gx; go[1] = gy; go[2] = gz;
            }
            if (lap_out) lap_out[(size_t)w * nel + i] = lp;
            if (one_out) one_out[(size_t)w * nel + i] = one;
            ek += lp;
        }
        if (ekin_out) ekin_out[w] = -0.5 * ek;
    }
    free(v);
    return rc;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
