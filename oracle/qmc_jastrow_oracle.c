/*
 * qmc_jastrow_oracle.c -- TEST INFRASTRUCTURE.  Plain, slow, fp64 CPU oracle for the Jastrow factor
 * of arxiv 1802.06922 (sec 7), as far as the particle-by-particle move needs it:
 * the value J and the ratio Psi(R')/Psi(R) = exp(-(J(R') - J(R))) of a single-electron move.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
 * load or call this file.  It shares no code, header, table or helper with the CUDA path.
 *
 * What it computes, and the passage each function follows ("R:Ax" = a reading in DESIGN.md sec 3):
 *
 *   orc_b3             eq. 33 (L369-373): "B_3(x) denotes a cardinal cubic B-spline function defined
 *                      on the interval x in [-3, 1) (centered at x = -1)": the four cubic pieces of the
 *                      uniform B-spline with knots -3,-2,-1,0,1, written out.
 *   orc_jastrow_u      eq. 33:  u(r) = sum_{m=0}^{M} p_m B_3(r / (r_c / M) - m), the literal sum over
 *                      ALL M+1 control points; u = 0 for r >= r_c ("r_c is the cutoff radius") (R:A21).
 *   orc_min_image      L375 "in periodic boundary conditions the cutoffs must be smaller than the
 *                      simulation cell Wigner-Seitz radius": a pair interacts through its nearest image
 *                      only; found by brute force over the (2 range + 1)^3 lattice translations around
 *                      the image that rounding the reduced coordinates gives.
 *   orc_jastrow_value  eq. 30 truncated after the two-body term, eq. 31, eq. 32 first term:
 *                      J = sum_i sum_I u_{I}(|r_i - R_I|) + 1/2 sum_{i != j} u_{s_i s_j}(|r_i - r_j|)
 *                      with "the up-up and down-down terms ... constrained to be equal" (L365): one
 *                      same-spin and one opposite-spin function.
 *   orc_jastrow_dj     the terms of J that contain electron k, at r' minus at r_k: what the move of ONE
 *                      electron changes (L195 particle-by-particle moves).  Psi'/Psi gains the factor
 *                      exp(-dJ) since Psi = e^{-J} Phi (eq. 28, eq. 29).
 *
 * The electrons of ONE sweep are the first argument (same spin among themselves, function f_same);
 * everything that stays fixed during that sweep is a CENTRE with a function of its own: the ions
 * (shared by all walkers, eq. 31) and the electrons of the other spin (per walker, function f_opp).
 *
 * Function table: nfunc functions; function f has cutoff rc[f], M[f] intervals and M[f] + 1 control
 * points p[poff[f] .. poff[f] + M[f]].  An index of -1 means "no such term".
 */
#include <math.h>
#include <stddef.h>

/* eq. 33: cardinal cubic B-spline with support [-3, 1), centred at x = -1. */
double orc_b3(double x)
{
    double y = x + 3.0; /* knots 0,1,2,3,4 */
    if (!(y >= 0.0) || y >= 4.0) return 0.0;
    if (y < 1.0) return y * y * y / 6.0;
    if (y < 2.0) { double t = y - 1.0; return (-3.0 * t * t * t + 3.0 * t * t + 3.0 * t + 1.0) / 6.0; }
    if (y < 3.0) { double t = y - 2.0; return (3.0 * t * t * t - 6.0 * t * t + 4.0) / 6.0; }
    { double t = 4.0 - y; return t * t * t / 6.0; }
}

/* eq. 33, every term of the sum; zero at and beyond the cutoff. */
double orc_jastrow_u(double r, double rc, int M, const double *p)
{
    if (M <= 0 || !(rc > 0.0) || !(r < rc) || r < 0.0) return r != r ? r : 0.0; /* NaN in, NaN out */
    double delta = rc / (double)M, s = 0.0;
    for (int m = 0; m <= M; ++m) s += p[m] * orc_b3(r / delta - (double)m);
    return s;
}

static int inv3j(const double L[9], double Li[9])
{
    double det = L[0] * (L[4] * L[8] - L[5] * L[7]) - L[1] * (L[3] * L[8] - L[5] * L[6]) +
                 L[2] * (L[3] * L[7] - L[4] * L[6]);
    if (det == 0.0 || !isfinite(det)) return -1;
    /* adjugate / det, row by row */
    Li[0] = (L[4] * L[8] - L[5] * L[7]) / det;
    Li[1] = (L[2] * L[7] - L[1] * L[8]) / det;
    Li[2] = (L[1] * L[5] - L[2] * L[4]) / det;
    Li[3] = (L[5] * L[6] - L[3] * L[8]) / det;
    Li[4] = (L[0] * L[8] - L[2] * L[6]) / det;
    Li[5] = (L[2] * L[3] - L[0] * L[5]) / det;
    Li[6] = (L[3] * L[7] - L[4] * L[6]) / det;
    Li[7] = (L[1] * L[6] - L[0] * L[7]) / det;
    Li[8] = (L[0] * L[4] - L[1] * L[3]) / det;
    return 0;
}

/* Distance between a and b under periodic boundary conditions: the smallest |a - b + m . lattice|
 * over integer m within `range` of the image that rounding the reduced coordinates gives.
 * lattice == NULL: open boundary conditions, the plain distance. */
double orc_min_image(const double *lattice, const double a[3], const double b[3], int range)
{
    double d[3] = {a[0] - b[0], a[1] - b[1], a[2] - b[2]};
    if (!lattice) return sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double Li[9];
    if (inv3j(lattice, Li)) return NAN;
    double u[3];
    for (int c = 0; c < 3; ++c) {
        u[c] = d[0] * Li[0 * 3 + c] + d[1] * Li[1 * 3 + c] + d[2] * Li[2 * 3 + c];
        u[c] -= floor(u[c] + 0.5);
    }
    double best = INFINITY;
    for (int i = -range; i <= range; ++i)
        for (int j = -range; j <= range; ++j)
            for (int k = -range; k <= range; ++k) {
                double v[3] = {u[0] + i, u[1] + j, u[2] + k}, x[3];
                for (int c = 0; c < 3; ++c) x[c] = v[0] * lattice[0 * 3 + c] + v[1] * lattice[1 * 3 + c] + v[2] * lattice[2 * 3 + c];
                double r = sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
                if (r < best || r != r) best = r;
            }
    return best;
}

typedef struct orc_jastrow {
    int nfunc;
    const double *rc;   /* [nfunc] */
    const int *M;       /* [nfunc] */
    const int *poff;    /* [nfunc] */
    const double *p;    /* control points, concatenated */
    int f_same, f_opp;  /* electron-electron functions (-1: none) */
    const double *lattice; /* 9 doubles or NULL (open boundaries) */
    int nion;
    const double *ion;  /* [nion][3] */
    const int *ion_func;/* [nion] */
    int range;          /* images searched per dimension around the rounded one (>= 1) */
} orc_jastrow;

static double u_of(const orc_jastrow *J, int f, double r)
{
    if (f < 0 || f >= J->nfunc) return 0.0;
    return orc_jastrow_u(r, J->rc[f], J->M[f], J->p + J->poff[f]);
}

/* eq. 30 (one- and two-body terms) for ONE walker: nel electrons of one spin at pos, nother electrons
 * of the other spin at other.  The other-spin electrons' own same-spin and electron-ion terms are
 * included, so this is the J of the whole configuration. */
double orc_jastrow_value(const orc_jastrow *J, int nel, const double *pos, int nother, const double *other)
{
    double s = 0.0;
    for (int i = 0; i < nel; ++i)
        for (int I = 0; I < J->nion; ++I)
            s += u_of(J, J->ion_func[I], orc_min_image(J->lattice, pos + 3 * i, J->ion + 3 * I, J->range));
    for (int i = 0; i < nother; ++i)
        for (int I = 0; I < J->nion; ++I)
            s += u_of(J, J->ion_func[I], orc_min_image(J->lattice, other + 3 * i, J->ion + 3 * I, J->range));
    /* 1/2 sum over ordered pairs i != j */
    double s2 = 0.0;
    for (int i = 0; i < nel + nother; ++i)
        for (int j = 0; j < nel + nother; ++j) {
            if (i == j) continue;
            const double *a = i < nel ? pos + 3 * i : other + 3 * (i - nel);
            const double *b = j < nel ? pos + 3 * j : other + 3 * (j - nel);
            int same = (i < nel) == (j < nel);
            s2 += u_of(J, same ? J->f_same : J->f_opp, orc_min_image(J->lattice, a, b, J->range));
        }
    return s + 0.5 * s2;
}

/* J(electron k at rnew) - J(electron k at pos[k]), everything else fixed: the terms of eq. 30 that
 * contain electron k (electron-ion, same spin, opposite spin). */
double orc_jastrow_dj(const orc_jastrow *J, int nel, const double *pos, int nother, const double *other,
                      int k, const double rnew[3])
{
    const double *rk = pos + 3 * k;
    double d = 0.0;
    for (int I = 0; I < J->nion; ++I)
        d += u_of(J, J->ion_func[I], orc_min_image(J->lattice, rnew, J->ion + 3 * I, J->range)) -
             u_of(J, J->ion_func[I], orc_min_image(J->lattice, rk, J->ion + 3 * I, J->range));
    for (int j = 0; j < nel; ++j) {
        if (j == k) continue;
        d += u_of(J, J->f_same, orc_min_image(J->lattice, rnew, pos + 3 * j, J->range)) -
             u_of(J, J->f_same, orc_min_image(J->lattice, rk, pos + 3 * j, J->range));
    }
    for (int j = 0; j < nother; ++j)
        d += u_of(J, J->f_opp, orc_min_image(J->lattice, rnew, other + 3 * j, J->range)) -
             u_of(J, J->f_opp, orc_min_image(J->lattice, rk, other + 3 * j, J->range));
    return d;
}
