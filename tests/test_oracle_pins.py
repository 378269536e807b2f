"""Pins of the fp64 CPU oracle (oracle/qmc_oracle.c) against facts the paper's formulation
and the mathematics fix -- none of them re-types the oracle's own formulas:

  P-a  partition of unity (constant table)
  P-b  linear / P-c quadratic and bilinear reproduction (index offset of eq. 33;
       gradient and Laplacian scaling, incl. the cross terms on a skewed cell)
  P-d  plane-wave table: closed form at the grid nodes, across the periodic wrap
  P-e  periodicity, P-f C2 continuity across cell faces
  P-s  scipy.interpolate.BSpline tensor product (de Boor recursion, a library routine)
  P-g  central finite differences of the oracle's own value
  P-h  ratio vs Leibniz-expansion and numpy determinants (N <= 16)          L299, L325
  P-i  Sherman-Morrison vs numpy.linalg.inv of the row-replaced matrix      L299
  P-j  sweep: sum of log|R| over accepted moves telescopes to the LU log-det difference
  P-k  sweep: B_final^T A_final = I with A recomputed from the final positions
  P-m  accept control flow (u = 0, u -> 1, zero displacement)               L195-199, eq. 12
"""
import itertools
import math

import numpy as np
import pytest
from scipy.interpolate import BSpline

import oracle
from paper_1802_06922_b200 import inputs

SKEW = np.array([[3.1, 0.2, -0.1], [0.4, 2.7, 0.3], [-0.2, 0.5, 3.4]])
ORTHO = np.diag([2.4, 3.0, 3.5])


def rand_table(rng, grid, norb):
    return rng.uniform(-1, 1, size=(*grid, norb)).astype(np.float32)


def grid_coords(lat, grid, pos):
    """Reduced grid coordinates s in [0, N_d) and J[j][d] = d s_d / d r_j, via numpy only."""
    li = np.linalg.inv(lat)
    u = pos @ li
    u = u - np.floor(u)
    s = u * np.asarray(grid, dtype=np.float64)
    J = li * np.asarray(grid, dtype=np.float64)[None, :]
    return s, J


# ----------------------------------------------------------------------------- P-a
@pytest.mark.parametrize("lat", [ORTHO, SKEW])
def test_partition_of_unity(lat):
    rng = np.random.default_rng(1)
    grid, norb = (7, 5, 6), 3
    coefs = np.empty((*grid, norb), dtype=np.float32)
    coefs[..., 0], coefs[..., 1], coefs[..., 2] = 0.75, -2.5, 1.0
    pos = rng.uniform(-2, 2, size=(50, 3)) @ lat
    v, g, l = oracle.spline_vgl(coefs, lat, pos)
    assert np.allclose(v, np.array([0.75, -2.5, 1.0])[None, :], atol=1e-14)
    assert np.max(np.abs(g)) < 1e-13
    assert np.max(np.abs(l)) < 1e-12


# ----------------------------------------------------------------------------- P-b, P-c
@pytest.mark.parametrize("lat", [ORTHO, SKEW])
def test_polynomial_reproduction(lat):
    """c = alpha + beta*ix -> phi = alpha + beta*(s_x + 1): control point m is supported on
    [m-3, m+1) (eq. 33's convention), so the spline of c_i = i is s + 1.  c = ix^2 ->
    (s_x+1)^2 + 1/3.  c = ix*iy -> (s_x+1)(s_y+1)."""
    rng = np.random.default_rng(2)
    grid = (16, 14, 12)
    ix = np.arange(grid[0], dtype=np.float64)[:, None, None]
    iy = np.arange(grid[1], dtype=np.float64)[None, :, None]
    one = np.ones(grid)
    alpha, beta = 0.5, 0.25
    coefs = np.stack([alpha + beta * ix * one, ix * ix * one, ix * iy * one,
                      (iy * iy * one)], axis=-1).astype(np.float32)
    # stay away from the periodic wrap: s_d in [0, N_d - 4)
    sfrac = rng.uniform(0, 1, size=(60, 3)) * (np.array(grid) - 4.0)
    pos = (sfrac / np.array(grid)) @ lat
    s, J = grid_coords(lat, grid, pos)
    v, g, l = oracle.spline_vgl(coefs, lat, pos)
    sx, sy = s[:, 0], s[:, 1]
    assert np.allclose(v[:, 0], alpha + beta * (sx + 1), atol=1e-12)
    assert np.allclose(v[:, 1], (sx + 1) ** 2 + 1.0 / 3.0, atol=1e-11)
    assert np.allclose(v[:, 2], (sx + 1) * (sy + 1), atol=1e-11)
    # gradients: d/dr_j = sum_d J[j][d] d/ds_d
    for j in range(3):
        assert np.allclose(g[:, j, 0], beta * J[j, 0], atol=1e-12)
        assert np.allclose(g[:, j, 1], 2 * (sx + 1) * J[j, 0], atol=1e-10)
        assert np.allclose(g[:, j, 2], (sy + 1) * J[j, 0] + (sx + 1) * J[j, 1], atol=1e-10)
    assert np.max(np.abs(l[:, 0])) < 1e-11
    assert np.allclose(l[:, 1], 2.0 * np.dot(J[:, 0], J[:, 0]), atol=1e-9)
    assert np.allclose(l[:, 2], 2.0 * np.dot(J[:, 0], J[:, 1]), atol=1e-9)   # cross term
    assert np.allclose(l[:, 3], 2.0 * np.dot(J[:, 1], J[:, 1]), atol=1e-9)


def test_orthorhombic_gradient_scale():
    """On an orthorhombic cell d/dx = (Nx/Lx) d/ds_x exactly."""
    grid, L = (10, 10, 10), np.array([2.0, 4.0, 5.0])
    iz = np.arange(10, dtype=np.float64)[None, None, :] * np.ones(grid)
    coefs = iz[..., None].astype(np.float32)
    pos = np.array([[0.3, 0.7, 1.1], [1.2, 3.3, 2.2]])
    v, g, l = oracle.spline_vgl(coefs, np.diag(L), pos)
    assert np.allclose(g[:, 2, 0], 10 / 5.0, atol=1e-13)
    assert np.allclose(g[:, :2, 0], 0.0, atol=1e-13)
    assert np.allclose(v[:, 0], pos[:, 2] / 5.0 * 10 + 1.0, atol=1e-13)


# ----------------------------------------------------------------------------- P-d
def test_planewave_nodes_closed_form():
    """c = cos(kappa.i + theta), kappa_d = 2 pi n_d / N_d.  At the grid nodes (t = 0) the cubic
    B-spline weights are (1,4,1,0)/6, whence phi = prod_d (2+cos kappa_d)/3 * cos(psi),
    psi = kappa.(i+1) + theta;  d/ds_x -> -sin(kappa_x) * (...) sin(psi);
    d2/ds_x2 -> 2(cos kappa_x - 1) (...) cos(psi).  Includes nodes that wrap in x and z."""
    grid = (16, 12, 20)
    nvec, theta = np.array([3, -2, 5]), 0.7
    kap = 2 * np.pi * nvec / np.array(grid)
    I = np.stack(np.meshgrid(*[np.arange(n) for n in grid], indexing="ij"), axis=-1)
    coefs = np.cos(I @ kap + theta)[..., None].astype(np.float32)
    cd = coefs[..., 0].astype(np.float64)          # the exact fp32 bits the oracle sees
    lat = ORTHO
    nodes = np.array([[2, 3, 4], [15, 5, 19], [14, 11, 18], [13, 0, 17], [0, 0, 0]])
    pos = (nodes / np.array(grid)) @ lat
    v, g, l = oracle.spline_vgl(coefs, lat, pos)
    s, J = grid_coords(lat, grid, pos)
    al = (2 + np.cos(kap)) / 3
    for p, nd in enumerate(nodes):
        psi = kap @ (nd + 1) + theta
        phi = al.prod() * np.cos(psi)
        # fp32 rounding of the table bounds the mismatch: |dc| <= 6e-8
        assert abs(v[p, 0] - phi) < 2e-7
        d1 = np.array([-np.sin(kap[d]) * al.prod() / al[d] * np.sin(psi) for d in range(3)])
        d2 = np.array([2 * (np.cos(kap[d]) - 1) * al.prod() / al[d] * np.cos(psi) for d in range(3)])
        assert np.allclose(g[p, :, 0], J @ d1, atol=2e-6)
        assert abs(l[p, 0] - np.sum(np.diag(J) ** 2 * d2)) < 2e-5
        # and exactly (to rounding) from the fp32 table itself with the node weights
        w = np.array([1, 4, 1]) / 6.0
        acc = 0.0
        for a, b, c in itertools.product(range(3), repeat=3):
            acc += w[a] * w[b] * w[c] * cd[(nd[0] + a) % 16, (nd[1] + b) % 12, (nd[2] + c) % 20]
        assert abs(v[p, 0] - acc) < 1e-14


def test_planewave_general_t_closed_form():
    """Same table at GENERAL fractions t (the closed form of SURVEY P-d): with weights b_a(t_d),
    phi = Re[ e^{i(kappa.i + theta)} prod_d sum_a b_a(t_d) e^{i kappa_d a} ], where the b_a are taken
    from scipy's de Boor recursion (not from the oracle's polynomials); first s-derivatives likewise
    with scipy's derivative basis.  Positions include cells that wrap in x and z."""
    grid = (16, 12, 20)
    nvec, theta = np.array([3, -2, 5]), 0.7
    kap = 2 * np.pi * nvec / np.array(grid)
    I = np.stack(np.meshgrid(*[np.arange(n) for n in grid], indexing="ij"), axis=-1)
    exact = np.cos(I @ kap + theta)
    coefs = exact[..., None].astype(np.float32)
    lat = SKEW
    rng = np.random.default_rng(21)
    cells = np.array([[2, 3, 4], [15, 5, 19], [14, 11, 18], [13, 0, 17], [0, 0, 0], [15, 11, 19]])
    tt = rng.uniform(0.02, 0.98, size=cells.shape)
    pos = ((cells + tt) / np.array(grid)) @ lat
    v, g, l = oracle.spline_vgl(coefs, lat, pos)
    s, J = grid_coords(lat, grid, pos)
    for p, (nd, t) in enumerate(zip(cells, tt)):
        assert np.allclose(s[p], nd + t, atol=1e-9)
        fac, dfac = [], []
        for d in range(3):
            b = _scipy_basis(grid[d], np.array([nd[d] + t[d]]), 0)[0]      # weights of control points by index
            db = _scipy_basis(grid[d], np.array([nd[d] + t[d]]), 1)[0]
            ph = np.exp(1j * kap[d] * np.arange(grid[d] + 3))     # extended control points m = 0..n+2
            fac.append(np.sum(b * ph))
            dfac.append(np.sum(db * ph))
        e0 = np.exp(1j * theta)
        phi = (e0 * fac[0] * fac[1] * fac[2]).real
        d1 = np.array([(e0 * dfac[0] * fac[1] * fac[2]).real, (e0 * fac[0] * dfac[1] * fac[2]).real,
                       (e0 * fac[0] * fac[1] * dfac[2]).real])
        assert abs(v[p, 0] - phi) < 2e-7          # fp32 rounding of the table: |dc| <= 6e-8
        assert np.allclose(g[p, :, 0], J @ d1, atol=5e-6)


def test_cell_face_rounding_and_nonfinite_positions():
    """R:A7 / R:A18.  A reduced coordinate that rounds UP to 1.0 (r = -1e-18 a0: u = -tiny,
    u - floor(u) = 1.0 in fp64) is the point u = 0: cell 0, t = 0, the same bits as r = 0, and the
    node weights (1,4,1,0)/6 applied to control points 0,1,2 give the value.  A non-finite position
    gives NaN orbitals (never an out-of-range table read)."""
    rng = np.random.default_rng(3)
    grid, norb = (6, 5, 7), 4
    coefs = rand_table(rng, grid, norb)
    for lat in (ORTHO, SKEW):
        for d in range(3):
            eps = -1e-18 * lat[d]
            u = eps @ np.linalg.inv(lat)
            assert (u[d] - np.floor(u[d])) == 1.0                      # the case is really exercised
            v, g, l = oracle.spline_vgl(coefs, lat, np.stack([eps, np.zeros(3), lat[d]]))
            assert np.array_equal(v[0], v[1]) or np.max(np.abs(v[0] - v[1])) < 1e-15
            assert np.max(np.abs(v[0] - v[2])) < 1e-14 and np.max(np.abs(g[0] - g[1])) < 1e-12
            assert np.max(np.abs(l[0] - l[1])) < 1e-10
        w = np.array([1, 4, 1]) / 6.0
        cd = coefs.astype(np.float64)
        ref = np.einsum("a,b,c,abcn->n", w, w, w, cd[:3, :3, :3])
        v0 = oracle.spline_vgl(coefs, lat, np.zeros((1, 3)), want_gl=False)
        assert np.max(np.abs(v0[0] - ref)) < 1e-15
    for bad in (np.nan, np.inf, -np.inf):
        v, g, l = oracle.spline_vgl(coefs, ORTHO, np.array([[0.3, bad, 0.1]]))
        assert np.isnan(v).all() and np.isnan(g).all() and np.isnan(l).all()


# ----------------------------------------------------------------------------- P-e, P-f
def test_periodicity_and_continuity():
    rng = np.random.default_rng(3)
    grid, norb = (6, 7, 5), 4
    coefs = rand_table(rng, grid, norb)
    lat = SKEW
    pos = rng.uniform(0, 1, size=(20, 3)) @ lat
    v0, g0, l0 = oracle.spline_vgl(coefs, lat, pos)
    shift = np.array([[1, 0, 0], [0, -2, 1], [3, 1, -1]]) @ lat
    for sh in shift:
        v1, g1, l1 = oracle.spline_vgl(coefs, lat, pos + sh)
        assert np.max(np.abs(v1 - v0)) < 1e-12
        assert np.max(np.abs(g1 - g0)) < 1e-10
        assert np.max(np.abs(l1 - l0)) < 1e-8
    # C2 continuity across every cell face, incl. the periodic one (value, grad, lap)
    eps = 1e-9
    for d in range(3):
        for face in range(grid[d] + 1):
            u = rng.uniform(0.05, 0.95, size=3)
            u[d] = face / grid[d]
            um, up = u.copy(), u.copy()
            um[d] -= eps / grid[d]
            up[d] += eps / grid[d]
            vm, gm, lm = oracle.spline_vgl(coefs, lat, (um @ lat)[None])
            vp, gp, lp = oracle.spline_vgl(coefs, lat, (up @ lat)[None])
            assert np.max(np.abs(vm - vp)) < 1e-7
            assert np.max(np.abs(gm - gp)) < 1e-6
            assert np.max(np.abs(lm - lp)) < 1e-4     # third derivative jumps: O(eps) gap


# ----------------------------------------------------------------------------- P-s
def _scipy_basis(n, s, nu):
    """All basis values (nu-th derivative) of the uniform cubic B-spline with control point m
    supported on [m-3, m+1): knots t_j = j - 3.  Returns [npts][n+3] for extended control
    points m = 0..n+2 (m >= n wraps to m - n)."""
    ncoef = n + 3
    t = np.arange(-3, ncoef + 1, dtype=np.float64)
    return BSpline(t, np.eye(ncoef), 3)(s, nu=nu)


@pytest.mark.parametrize("lat", [ORTHO, SKEW])
def test_against_scipy_bspline(lat):
    rng = np.random.default_rng(4)
    grid, norb = (6, 5, 7), 5
    coefs = rand_table(rng, grid, norb)
    pos = rng.uniform(-1, 2, size=(80, 3)) @ lat          # also outside the home cell
    s, J = grid_coords(lat, grid, pos)
    ext = coefs.astype(np.float64)
    ext = np.concatenate([ext, ext[:3]], axis=0)
    ext = np.concatenate([ext, ext[:, :3]], axis=1)
    ext = np.concatenate([ext, ext[:, :, :3]], axis=2)
    Bs = [[_scipy_basis(grid[d], s[:, d], nu) for nu in range(3)] for d in range(3)]

    def contract(nx_, ny_, nz_):
        return np.einsum("pi,pj,pk,ijkn->pn", Bs[0][nx_], Bs[1][ny_], Bs[2][nz_], ext)

    v_ref = contract(0, 0, 0)
    d1 = np.stack([contract(1, 0, 0), contract(0, 1, 0), contract(0, 0, 1)], axis=1)   # [p][d][n]
    H = np.empty((len(pos), 3, 3, norb))
    orders = {(0, 0): (2, 0, 0), (1, 1): (0, 2, 0), (2, 2): (0, 0, 2),
              (0, 1): (1, 1, 0), (0, 2): (1, 0, 1), (1, 2): (0, 1, 1)}
    for (d, e), o in orders.items():
        H[:, d, e] = H[:, e, d] = contract(*o)
    g_ref = np.einsum("jd,pdn->pjn", J, d1)
    l_ref = np.einsum("jd,je,pden->pn", J, J, H)
    v, g, l = oracle.spline_vgl(coefs, lat, pos)
    assert np.max(np.abs(v - v_ref)) < 1e-13
    assert np.max(np.abs(g - g_ref)) < 1e-12
    assert np.max(np.abs(l - l_ref)) < 1e-11


# ----------------------------------------------------------------------------- P-g
def test_finite_differences():
    x = inputs.make_inputs(inputs.custom_config("fd", (12, 10, 14), 6, SKEW * 2.0, nw=4))
    coefs, lat = x.coefs_numpy(), x.lattice
    pos = x.pos.reshape(-1, 3)[:12]
    v, g, l = oracle.spline_vgl(coefs, lat, pos)
    h = 1e-4 * 0.4
    lap_fd = np.zeros_like(l)
    for j in range(3):
        e = np.zeros(3)
        e[j] = h
        vp = oracle.spline_vgl(coefs, lat, pos + e, want_gl=False)
        vm = oracle.spline_vgl(coefs, lat, pos - e, want_gl=False)
        gfd = (vp - vm) / (2 * h)
        assert np.max(np.abs(gfd - g[:, j, :])) < 1e-7 * max(1.0, np.max(np.abs(g)))
        lap_fd += (vp - 2 * v + vm) / (h * h)
    assert np.max(np.abs(lap_fd - l)) < 1e-5 * max(1.0, np.max(np.abs(l)))


# ----------------------------------------------------------------------------- P-h, P-i, LU
def _leibniz_det(A):
    n = A.shape[0]
    tot = 0.0
    for perm in itertools.permutations(range(n)):
        sgn = 1
        for i in range(n):
            for j in range(i + 1, n):
                if perm[i] > perm[j]:
                    sgn = -sgn
        tot += sgn * math.prod(A[i, perm[i]] for i in range(n))
    return tot


@pytest.mark.parametrize("n", [1, 2, 3, 5, 6])
def test_ratio_vs_leibniz(n):
    rng = np.random.default_rng(10 + n)
    A = rng.normal(size=(n, n))
    B, ld, sg = oracle.binv_from_A(A)
    d0 = _leibniz_det(A)
    assert abs(sg * math.exp(ld) - d0) < 1e-12 * max(1, abs(d0))
    for k in range(n):
        phi = rng.normal(size=n)
        A2 = A.copy()
        A2[k] = phi
        assert abs(oracle.det_ratio(B, k, phi) - _leibniz_det(A2) / d0) < 1e-10 * max(1, abs(_leibniz_det(A2) / d0))


@pytest.mark.parametrize("n", [4, 11, 16])
def test_ratio_and_sm_vs_numpy(n):
    rng = np.random.default_rng(20 + n)
    A = rng.normal(size=(n, n))
    B, ld, sg = oracle.binv_from_A(A)
    sgn_np, ld_np = np.linalg.slogdet(A)
    assert sg == int(sgn_np) and abs(ld - ld_np) < 1e-11
    assert np.max(np.abs(B.T - np.linalg.inv(A))) < 1e-10
    Ai, ld2, sg2 = oracle.lu_inverse(A)
    assert np.max(np.abs(Ai @ A - np.eye(n))) < 1e-11
    for k in [0, n // 2, n - 1]:
        phi = rng.normal(size=n)
        A2 = A.copy()
        A2[k] = phi
        R = oracle.det_ratio(B, k, phi)
        assert abs(R - np.linalg.det(A2) / np.linalg.det(A)) < 1e-9 * max(1, abs(R))
        B2 = oracle.sm_update(B, k, phi, R)
        assert np.max(np.abs(B2.T - np.linalg.inv(A2))) < 1e-8 * max(1.0, np.max(np.abs(B2)))
        # chain: keep moving from the updated state
        A, B = A2, B2


def test_sm_64_vs_direct_inverse():
    rng = np.random.default_rng(31)
    n = 64
    A = rng.normal(size=(n, n))
    B, _, _ = oracle.binv_from_A(A)
    for k in range(n):
        phi = rng.normal(size=n)
        R = oracle.det_ratio(B, k, phi)
        B = oracle.sm_update(B, k, phi, R)
        A[k] = phi
    assert np.max(np.abs(B.T - np.linalg.inv(A))) < 1e-9 * np.max(np.abs(B))


def test_lu_flags_singular():
    A = np.array([[1.0, 2.0, 3.0], [2.0, 4.0, 6.0], [0.0, 1.0, 1.0]])
    with pytest.raises(RuntimeError):
        oracle.lu_inverse(A)


def test_lu_needs_pivoting():
    A = np.array([[0.0, 1.0], [1.0, 0.0]])
    Ai, ld, sg = oracle.lu_inverse(A)
    assert sg == -1 and abs(ld) < 1e-15 and np.allclose(Ai, A)


# ----------------------------------------------------------------------------- sweeps
@pytest.fixture(scope="module")
def sweep_case():
    cfg = inputs.custom_config("sweep", (12, 10, 14), 24, SKEW * 2.0, nw=3, nsweeps=2, sigma=0.25)
    x = inputs.make_inputs(cfg)
    coefs = x.coefs_numpy()
    A = oracle.slater_matrix(coefs, x.lattice, x.pos)
    B = np.empty_like(A)
    ld = np.empty(cfg.nw)
    sg = np.empty(cfg.nw, dtype=np.int32)
    for w in range(cfg.nw):
        B[w], ld[w], sg[w] = oracle.binv_from_A(A[w])
    return x, coefs, A, B, ld, sg


def test_slater_matrix_layout(sweep_case):
    """A[w][i][j] = phi_j(r_wi) (L325): row = electron, column = orbital."""
    x, coefs, A, *_ = sweep_case
    v = oracle.spline_vgl(coefs, x.lattice, x.pos[1, 5][None], want_gl=False)
    assert np.array_equal(A[1, 5], v[0])


def test_sweep_telescoping_and_inverse(sweep_case):
    x, coefs, A, B, ld, sg = sweep_case
    out = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, A=A)
    acc = out["accept"].astype(bool)
    assert 0 < acc.sum() < acc.size
    A_fin = oracle.slater_matrix(coefs, x.lattice, out["pos"])
    assert np.max(np.abs(A_fin - out["A"])) < 1e-13
    for w in range(x.cfg.nw):
        s_np, l_np = np.linalg.slogdet(A_fin[w])
        s0, l0 = np.linalg.slogdet(A[w])
        tele = np.sum(np.log(np.abs(out["ratios"][..., w][acc[..., w]])))
        assert abs(tele - (l_np - l0)) < 1e-8
        assert abs(out["logdet"][w] - l_np) < 1e-8
        assert out["sign"][w] == int(s_np)
        res = out["B"][w].T @ A_fin[w] - np.eye(x.cfg.norb)
        assert np.max(np.sum(np.abs(res), axis=1)) < 1e-8
    # decisions follow eq. 12: accept iff R^2 > u
    assert np.array_equal(acc, out["ratios"] ** 2 > x.unif)
    # accepted electrons moved by exactly delta, rejected ones stayed
    moved = np.zeros_like(x.pos)
    for s in range(x.cfg.nsweeps):
        moved += np.where(acc[s].T[..., None], np.transpose(x.delta[s], (1, 0, 2)), 0.0)
    assert np.max(np.abs(out["pos"] - (x.pos + moved))) < 1e-14


def test_sweep_sm_equals_definitional(sweep_case):
    """Mode 0 (Sherman-Morrison) reaches the result of mode 1 (LU recompute after every
    accepted move) to rounding."""
    x, coefs, A, B, ld, sg = sweep_case
    o0 = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, A=A, mode=0)
    o1 = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, A=A, mode=1)
    assert np.array_equal(o0["accept"], o1["accept"])
    assert np.max(np.abs(o0["ratios"] - o1["ratios"])) < 1e-9
    assert np.max(np.abs(o0["B"] - o1["B"])) < 1e-9 * max(1.0, np.max(np.abs(o1["B"])))


def test_sweep_forced_and_replay(sweep_case):
    x, coefs, A, B, ld, sg = sweep_case
    free = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, A=A, want_phi=True)
    forced = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, 1.0 - x.unif, A=A,
                          forced=free["accept"])
    assert np.array_equal(forced["accept"], free["accept"])
    assert np.array_equal(forced["B"], free["B"]) and np.array_equal(forced["pos"], free["pos"])
    # replay of recorded orbital vectors (here rounded to fp32 -> small, nonzero change)
    phi32 = free["phi"].astype(np.float32)
    rep = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, forced=free["accept"],
                       phi_in=phi32)
    assert 0 < np.max(np.abs(rep["B"] - free["B"])) < 1e-4 * np.max(np.abs(free["B"]))
    # partial sweep: only the first 5 electrons are moved
    part = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta[:1], x.unif[:1], iel_count=5)
    assert np.array_equal(part["accept"][0, :5], free["accept"][0, :5])
    assert not part["accept"][0, 5:].any()
    assert np.array_equal(part["pos"][:, 5:], x.pos[:, 5:])


def test_accept_control_flow(sweep_case):
    x, coefs, A, B, ld, sg = sweep_case
    zeros = np.zeros_like(x.unif)
    out = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, zeros)
    assert out["accept"].all()                       # R != 0 w.p. 1  ->  R^2 > 0
    tot = np.transpose(x.delta.sum(axis=0), (1, 0, 2))
    assert np.max(np.abs(out["pos"] - (x.pos + tot))) < 1e-13
    ones = np.full_like(x.unif, 1.0 - 2.0 ** -53)
    out1 = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, ones)
    assert np.array_equal(out1["accept"].astype(bool), np.abs(out1["ratios"]) >= 1.0)
    # zero displacement: the new row equals the old one -> R = 1, B unchanged
    nod = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, np.zeros_like(x.delta), zeros)
    assert np.max(np.abs(nod["ratios"] - 1.0)) < 1e-10
    assert np.max(np.abs(nod["B"] - B)) < 1e-9 * np.max(np.abs(B))
    assert np.array_equal(nod["pos"], x.pos)
    # multi-threaded run gives the same bits (walkers are independent, L181)
    out_mt = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, nthreads=3)
    out_st = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, nthreads=1)
    assert np.array_equal(out_mt["B"], out_st["B"]) and np.array_equal(out_mt["ratios"], out_st["ratios"])


def test_sweep_singular_and_nonfinite_moves(sweep_case):
    """R:A8 / R:A18.  A NaN displacement gives a NaN ratio: rejected, nothing changes for that
    walker at that step.  An IMPOSED accept of a move with R = 0 (orbital vector identically zero)
    or NaN is refused: B, positions, log-det untouched; everything else proceeds as without it."""
    x, coefs, A, B, ld, sg = sweep_case
    delta = x.delta.copy()
    delta[0, 3, 1, 2] = np.nan
    out = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, delta[:1], np.zeros_like(x.unif[:1]), iel_count=4)
    assert np.isnan(out["ratios"][0, 3, 1]) and out["accept"][0, 3, 1] == 0
    assert out["accept"][0, :3].all() and out["accept"][0, 3, [0, 2]].all()
    assert np.array_equal(out["pos"][1, 3], x.pos[1, 3]) and np.isfinite(out["B"]).all()
    ref = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta[:1], np.zeros_like(x.unif[:1]), iel_count=3)
    assert np.array_equal(out["B"][1], ref["B"][1]) and out["logdet"][1] == ref["logdet"][1]
    # forced accept of R == 0 and of R = NaN
    nel, nw = x.cfg.norb, x.cfg.nw
    phi = np.ascontiguousarray(oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta[:1], x.unif[:1],
                                            want_phi=True)["phi"].astype(np.float32))
    phi[0, 2, 0, :] = 0.0
    phi[0, 4, 2, 5] = np.nan
    forced = np.ones((1, nel, nw), dtype=np.uint8)
    out = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta[:1], x.unif[:1], forced=forced, phi_in=phi)
    assert out["ratios"][0, 2, 0] == 0.0 and out["accept"][0, 2, 0] == 0
    assert np.isnan(out["ratios"][0, 4, 2]) and out["accept"][0, 4, 2] == 0
    assert out["accept"].sum() == nel * nw - 2
    assert np.isfinite(out["B"]).all() and np.isfinite(out["logdet"]).all()
    assert np.array_equal(out["pos"][0, 2], x.pos[0, 2]) and np.array_equal(out["pos"][2, 4], x.pos[2, 4])


def test_init_walkers_matches_numpy(sweep_case):
    x, coefs, A, B, ld, sg = sweep_case
    B2, ld2, sg2, A2 = oracle.init_walkers(coefs, x.lattice, x.pos, nthreads=2, want_A=True)
    assert np.array_equal(A2, A) and np.array_equal(B2, B) and np.array_equal(ld2, ld) and np.array_equal(sg2, sg)
    for w in range(x.cfg.nw):
        assert np.max(np.abs(B2[w].T - np.linalg.inv(A[w]))) < 1e-9 * np.max(np.abs(B2[w]))


def test_bnorm_diagnostic(sweep_case):
    """bnorm_out is the 1-norm of the row the ratio used: for the first move of walker w that is
    row 0 of the initial inverse."""
    x, coefs, A, B, ld, sg = sweep_case
    out = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, want_bnorm=True)
    for w in range(x.cfg.nw):
        assert abs(out["bnorm"][0, 0, w] - np.sum(np.abs(B[w, 0]))) < 1e-12
    # |R - R'| <= bnorm * max|phi - phi'| for any perturbed orbital vector
    assert np.all(out["bnorm"] > 0)


def test_wavefunction_force_against_finite_differences(sweep_case):
    """F = 2 grad log Psi_T (the F of eq. 11/13) of the moved electron at the proposed
    configuration.  Pin independent of the oracle's formula: F R / 2 = grad_r' (det A'(r') / det A),
    a smooth function of r' even next to a node (where F itself diverges), against central finite
    differences of that determinant ratio taken by numpy from Slater matrices at shifted positions
    (the walk is followed with the oracle's own decisions so the configuration is known)."""
    x, coefs, A, B, ld, sg = sweep_case
    out = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, want_force=True)
    F, acc = out["force"], out["accept"]
    assert np.isfinite(F).all() and np.abs(F).max() > 1e-3
    nsw, nel, nw = x.unif.shape
    h = 1e-5
    checked = 0
    for w in range(nw):
        pos = x.pos[w].copy()
        for s in range(nsw):
            for k in range(nel):
                rnew = pos[k] + x.delta[s, k, w]
                if (s * nel + k) % 7 == w:            # a sample of moves, accepted and rejected ones
                    s0, l0 = np.linalg.slogdet(oracle.slater_matrix(coefs, x.lattice, pos[None])[0])
                    fd = np.zeros(3)
                    for d in range(3):
                        val = []
                        for sgn in (+1.0, -1.0):
                            trial = pos.copy()
                            trial[k] = rnew
                            trial[k, d] += sgn * h
                            s1, l1 = np.linalg.slogdet(oracle.slater_matrix(coefs, x.lattice, trial[None])[0])
                            val.append(s1 * s0 * np.exp(l1 - l0))
                        fd[d] = (val[0] - val[1]) / (2.0 * h)
                    got = 0.5 * F[s, k, w] * out["ratios"][s, k, w]
                    scale = max(1.0, np.abs(fd).max())
                    assert np.max(np.abs(got - fd)) < 1e-6 * scale, (s, k, w, got, fd)
                    checked += 1
                if acc[s, k, w]:
                    pos[k] = rnew
    assert checked >= 15


def test_fixed_node_rule(sweep_case):
    """moves that change the sign of the wavefunction are rejected.  With u = 0 every
    move with R > 0 is accepted and every move with R < 0 rejected, so the sign of det A never
    changes and log|det| telescopes over the accepted (positive) ratios; where the free run met no
    negative ratio the flag changes nothing."""
    x, coefs, A, B, ld, sg = sweep_case
    zeros = np.zeros_like(x.unif)
    fn = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, zeros, A=A, fixed_node=True)
    assert np.array_equal(fn["accept"].astype(bool), fn["ratios"] > 0.0)
    assert (fn["ratios"] < 0.0).any(), "the case should propose at least one nodal crossing"
    assert np.array_equal(fn["sign"], sg)
    for w in range(x.pos.shape[0]):
        s_np, ld_np = np.linalg.slogdet(fn["A"][w])
        assert s_np == sg[w] and abs(ld_np - fn["logdet"][w]) < 1e-9
    free = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif)
    fixed = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, fixed_node=True)
    for w in range(x.pos.shape[0]):
        neg = (free["ratios"][:, :, w] < 0.0) & free["accept"][:, :, w].astype(bool)
        if not neg.any():
            assert np.array_equal(free["ratios"][:, :, w], fixed["ratios"][:, :, w])
        else:
            assert (fixed["ratios"][:, :, w][fixed["accept"][:, :, w].astype(bool)] > 0.0).all()


def test_det_kinetic_against_finite_differences(sweep_case):
    """Kinetic term of the local energy of Psi = det A (eq. 3 first term, eq. 37):
    grad_i det / det and lap_i det / det for every electron.  Pin independent of the cofactor formula:
    first and second central differences of det A(r_i +- h e_d) / det A with the determinants taken
    by numpy from Slater matrices at shifted positions; plus sum_j phi_j(r_i) B[i][j] = 1."""
    x, coefs, A, B, ld, sg = sweep_case
    out = oracle.det_kinetic(coefs, x.lattice, x.pos, B)
    assert np.max(np.abs(out["one"] - 1.0)) < 1e-10
    assert np.allclose(out["ekin"], -0.5 * out["lap"].sum(axis=1), rtol=0, atol=1e-9 * np.abs(out["lap"]).sum())
    nw, nel, _ = x.pos.shape
    h = 2e-4
    for w in range(nw):
        s0, l0 = np.linalg.slogdet(oracle.slater_matrix(coefs, x.lattice, x.pos[w][None])[0])
        for i in range(0, nel, 5):
            grad_fd, lap_fd = np.zeros(3), 0.0
            for d in range(3):
                r = []
                for sgn in (+1.0, -1.0):
                    trial = x.pos[w].copy()
                    trial[i, d] += sgn * h
                    s1, l1 = np.linalg.slogdet(oracle.slater_matrix(coefs, x.lattice, trial[None])[0])
                    r.append(s1 * s0 * np.exp(l1 - l0))
                grad_fd[d] = (r[0] - r[1]) / (2.0 * h)
                lap_fd += (r[0] - 2.0 + r[1]) / (h * h)
            gscale = max(1.0, np.abs(grad_fd).max())
            assert np.max(np.abs(out["grad"][w, i] - grad_fd)) < 1e-6 * gscale, (w, i, out["grad"][w, i], grad_fd)
            lscale = max(1.0, abs(lap_fd))
            assert abs(out["lap"][w, i] - lap_fd) < 2e-5 * lscale, (w, i, out["lap"][w, i], lap_fd)
    # a wrong inverse shows in `one`
    bad = oracle.det_kinetic(coefs, x.lattice, x.pos, np.roll(B, 1, axis=1))
    assert np.max(np.abs(bad["one"] - 1.0)) > 1e-3


# ----------------------------------------------------------------------------- drift moves (eq. 11-13)
def _logdet_at(coefs, lat, pos):
    s, l = np.linalg.slogdet(oracle.slater_matrix(coefs, lat, pos[None])[0])
    return s, l


def _fd_force(coefs, lat, pos, k, h=1e-5):
    """F_k = 2 grad_k log|det A| by central differences of numpy log-determinants (L156)."""
    f = np.zeros(3)
    for d in range(3):
        v = []
        for sgn in (+1.0, -1.0):
            t = pos.copy()
            t[k, d] += sgn * h
            v.append(_logdet_at(coefs, lat, t)[1])
        f[d] = 2.0 * (v[0] - v[1]) / (2.0 * h)
    return f


def test_drift_moves_against_closed_forms(sweep_case):
    """orc_sweep_ex with tau > 0.  Pins, none of them the oracle's own formulas:
    F_k(r) = 2 grad_k log|det A| at the CURRENT configuration against finite differences of numpy
    log-determinants; the proposal r' = r + tau F + chi (eq. 13 / eq. 19, lambda = 1/2); the
    transition ratio against scipy's Gaussian log-densities, T(r->r') = N(r'; r + tau F(r), tau I) and
    T(r'->r) = N(r; r' + tau F(r'), tau I) with F(r') again from finite differences at the proposed
    configuration; the decision rule of eq. 12; log-det telescoping and B^T A = I at the end."""
    from scipy.stats import multivariate_normal
    x, coefs, A, B, ld, sg = sweep_case
    tau = 0.02
    rng = np.random.default_rng(17)
    chi = rng.normal(0.0, np.sqrt(tau), size=x.delta.shape)
    out = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, chi, x.unif, A=A, tau=tau, want_force=True)
    acc = out["accept"].astype(bool)
    assert 0 < acc.sum() < acc.size
    assert np.array_equal(acc, out["ratios"] ** 2 * np.exp(out["logt"]) > x.unif)
    assert np.abs(out["logt"]).max() > 1e-3            # the ratio of the two Gaussians really matters
    nsw, nel, nw = x.unif.shape
    checked = 0
    for w in range(nw):
        pos = x.pos[w].copy()
        for s in range(nsw):
            for k in range(nel):
                rp = out["rprop"][s, k, w]
                assert np.max(np.abs(rp - (pos[k] + tau * out["fcur"][s, k, w] + chi[s, k, w]))) < 1e-14
                if (s * nel + k) % 9 == w:
                    f_cur = _fd_force(coefs, x.lattice, pos, k)
                    assert np.max(np.abs(out["fcur"][s, k, w] - f_cur)) < 1e-5 * max(1.0, np.abs(f_cur).max())
                    trial = pos.copy()
                    trial[k] = rp
                    if abs(out["ratios"][s, k, w]) > 0.05:      # FD of log|det| needs to stay off the node
                        f_new = _fd_force(coefs, x.lattice, trial, k)
                        fwd = multivariate_normal(mean=pos[k] + tau * f_cur, cov=tau * np.eye(3)).logpdf(rp)
                        bwd = multivariate_normal(mean=rp + tau * f_new, cov=tau * np.eye(3)).logpdf(pos[k])
                        assert abs(out["logt"][s, k, w] - (bwd - fwd)) < 2e-4 * max(1.0, abs(bwd - fwd)), (s, k, w)
                        checked += 1
                if acc[s, k, w]:
                    pos[k] = rp
        assert np.array_equal(pos, out["pos"][w])
        s_np, l_np = _logdet_at(coefs, x.lattice, out["pos"][w])
        assert abs(out["logdet"][w] - l_np) < 1e-8 and out["sign"][w] == int(s_np)
        res = out["B"][w].T @ oracle.slater_matrix(coefs, x.lattice, out["pos"][w][None])[0] - np.eye(nel)
        assert np.max(np.abs(res)) < 1e-8
    assert checked >= 8


def test_drift_reverse_move_identity(sweep_case):
    """Detailed balance structure: accept a move r -> r' (imposed), then propose the reverse move
    r' -> r from the new configuration (rprop_in): the determinant ratio is the reciprocal and the
    log transition ratio the negative of the forward one.  A swapped F(r) / F(r'), a wrong sign or a
    missing 1/R in the force at the proposal breaks this."""
    x, coefs, A, B, ld, sg = sweep_case
    tau = 0.03
    nsw, nel, nw = x.unif.shape
    chi = np.random.default_rng(5).normal(0.0, np.sqrt(tau), size=(1, nel, nw, 3))
    ones = np.ones((1, nel, nw), dtype=np.uint8)
    fwd = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, chi, x.unif[:1], forced=ones, tau=tau, iel_count=1,
                       want_force=True)
    back = oracle.sweep(coefs, x.lattice, fwd["pos"], fwd["B"], fwd["logdet"], fwd["sign"], chi, x.unif[:1],
                        forced=ones, tau=tau, iel_count=1,
                        rprop_in=np.broadcast_to(x.pos.transpose(1, 0, 2)[None], (1, nel, nw, 3)).copy())
    assert np.max(np.abs(back["ratios"][0, 0] * fwd["ratios"][0, 0] - 1.0)) < 1e-9
    assert np.max(np.abs(back["logt"][0, 0] + fwd["logt"][0, 0])) < 1e-8 * max(1.0, np.abs(fwd["logt"][0, 0]).max())
    assert np.max(np.abs(back["pos"] - x.pos)) == 0.0
    assert np.max(np.abs(back["B"] - B)) < 1e-8 * np.max(np.abs(B))
    # the force at the proposal of the forward move is the force at the current position of the reverse one
    assert np.max(np.abs(back["fcur"][0, 0] - fwd["force"][0, 0])) < 1e-8 * max(1.0, np.abs(fwd["force"][0, 0]).max())


def test_drift_small_tau_limit(sweep_case):
    """tau -> 0 with chi = sqrt(tau) z: the drift tau F and log T = O(sqrt(tau)) vanish against the
    diffusion, so the proposals tend to r + chi and the decisions to those of the no-drift walk
    (eq. 13 with F = 0) on the same displacements."""
    x, coefs, A, B, ld, sg = sweep_case
    z = np.random.default_rng(9).normal(size=x.delta.shape)
    tau = 1e-10
    chi = np.sqrt(tau) * z
    d = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, chi, x.unif, tau=tau)
    n = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, chi, x.unif)
    assert np.abs(d["logt"]).max() < 1e-2
    assert np.max(np.abs(d["ratios"] - n["ratios"])) < 1e-5
    same = d["accept"] == n["accept"]
    assert same.mean() > 0.99
    assert np.all(np.abs(n["ratios"][~same] ** 2 - x.unif[~same]) < 1e-2)


# ----------------------------------------------------------------------------- fp32-stored inverse (L82)
def test_fp32_stored_inverse(sweep_case):
    """R:A19.  b32 = 1: after every accepted move the stored inverse is the fp32 rounding of the fp64
    Sherman-Morrison result computed from the stored (fp32-valued) matrix -- checked move by move
    against orc_sm_update (itself pinned to numpy's inverse) followed by numpy's cast.  The residual
    B^T A - I sits at the fp32 level, grows slowly with the number of sweeps, and a recompute from the
    positions (orc_init_walkers) restores the fp64 level.  b32 = K (delayed rank-K storage) differs
    from b32 = 1 by a few fp32 ulps of max|B| only."""
    x, coefs, A, B, ld, sg = sweep_case
    nsw, nel, nw = x.unif.shape
    B32 = B.astype(np.float32).astype(np.float64)
    out = oracle.sweep(coefs, x.lattice, x.pos, B32, ld, sg, x.delta, x.unif, b32=1, want_phi=True)
    assert np.array_equal(out["B"], out["B"].astype(np.float32).astype(np.float64))
    # move-by-move replay with the pinned pieces
    for w in range(nw):
        Bw = B32[w].copy()
        for s in range(nsw):
            for k in range(nel):
                phi = out["phi"][s, k, w]
                R = oracle.det_ratio(Bw, k, phi)
                assert R == out["ratios"][s, k, w]
                if out["accept"][s, k, w]:
                    Bw = oracle.sm_update(Bw, k, phi, R).astype(np.float32).astype(np.float64)
        assert np.array_equal(Bw, out["B"][w])
    # residual level and growth, recompute
    delta4 = np.concatenate([x.delta, x.delta[::-1]], axis=0)
    unif4 = np.concatenate([x.unif, x.unif[::-1]], axis=0)
    o4 = oracle.sweep(coefs, x.lattice, x.pos, B32, ld, sg, delta4, unif4, b32=1)
    o1 = oracle.sweep(coefs, x.lattice, x.pos, B32, ld, sg, delta4[:1], unif4[:1], b32=1)
    o64 = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, delta4, unif4, forced=o4["accept"])

    def resid(Bm, pos):
        Af = oracle.slater_matrix(coefs, x.lattice, pos)
        return max(np.max(np.sum(np.abs(Bm[w].T @ Af[w] - np.eye(nel)), axis=1)) for w in range(nw))

    r1, r4, r64 = resid(o1["B"], o1["pos"]), resid(o4["B"], o4["pos"]), resid(o64["B"], o64["pos"])
    assert 1e-8 < r1 < 1e-3 and r4 < 1e-3 and r4 < 50.0 * r1 and r64 < 1e-9
    assert np.max(np.abs(o4["B"] - o64["B"])) < 1e-4 * np.max(np.abs(o64["B"]))
    Br, ldr, sgr = oracle.init_walkers(coefs, x.lattice, o4["pos"])
    assert resid(Br, o4["pos"]) < 1e-10
    assert np.max(np.abs(ldr - o4["logdet"])) < 1e-4 and np.array_equal(sgr, o4["sign"])
    # delayed-rank storage: same decisions here, and the stored matrices agree to a few fp32 ulps
    ok = oracle.sweep(coefs, x.lattice, x.pos, B32, ld, sg, x.delta, x.unif, b32=5, forced=out["accept"])
    assert np.array_equal(ok["B"], ok["B"].astype(np.float32).astype(np.float64))
    assert 0 < np.max(np.abs(ok["B"] - out["B"])) < 64 * 2.0 ** -24 * np.max(np.abs(out["B"]))
    # and b32 = K with a window that closes after every step is b32 = 1 exactly
    o_k1 = oracle.sweep(coefs, x.lattice, x.pos, B32, ld, sg, x.delta, x.unif, b32=1, forced=out["accept"])
    assert np.array_equal(o_k1["B"], out["B"])


# ----------------------------------------------------------------------------- D_up D_dn (eq. 26)
def test_wf_sweep_is_the_block_diagonal_determinant():
    """Psi_T = D_up D_dn (eq. 26 with one determinant per spin): oracle.wf_sweep (two
    independent sweeps) against numpy determinants of the BLOCK-DIAGONAL Slater matrix of all N_up + N_dn
    electrons: every ratio is det(M') / det(M) with the moved electron's row replaced, log|Psi| telescopes
    over the accepted moves, and an up move leaves the down block (and its inverse) untouched."""
    from scipy.linalg import block_diag
    cfgs = [inputs.custom_config("up", (10, 9, 11), 7, SKEW * 1.5, nw=2, nsweeps=2, sigma=0.3, index=201),
            inputs.custom_config("dn", (10, 9, 11), 5, SKEW * 1.5, nw=2, nsweeps=2, sigma=0.3, index=202)]
    xs = [inputs.make_inputs(c) for c in cfgs]
    spin = []
    for x in xs:
        coefs = x.coefs_numpy()
        B, ld, sg = oracle.init_walkers(coefs, x.lattice, x.pos)
        spin.append(dict(coefs=coefs, lattice=x.lattice, pos=x.pos, B=B, logdet=ld, sign=sg))
    nup, ndn, nw, nsw = 7, 5, 2, 2
    delta = np.concatenate([xs[0].delta, xs[1].delta], axis=1)
    unif = np.concatenate([xs[0].unif, xs[1].unif], axis=1)
    up, dn, ratios, accept = oracle.wf_sweep(spin, delta, unif)
    assert 0 < accept.sum() < accept.size

    def full_matrix(w, pu, pd):
        return block_diag(oracle.slater_matrix(spin[0]["coefs"], xs[0].lattice, pu[None])[0],
                          oracle.slater_matrix(spin[1]["coefs"], xs[1].lattice, pd[None])[0])

    for w in range(nw):
        pu, pd = xs[0].pos[w].copy(), xs[1].pos[w].copy()
        s0, l0 = np.linalg.slogdet(full_matrix(w, pu, pd))
        tele = 0.0
        for s_ in range(nsw):
            for k in range(nup + ndn):
                tu, td = pu.copy(), pd.copy()
                if k < nup:
                    tu[k] = pu[k] + delta[s_, k, w]
                else:
                    td[k - nup] = pd[k - nup] + delta[s_, k, w]
                sa, la = np.linalg.slogdet(full_matrix(w, pu, pd))
                sb, lb = np.linalg.slogdet(full_matrix(w, tu, td))
                brute = sa * sb * np.exp(lb - la)
                assert abs(ratios[s_, k, w] - brute) < 1e-8 * max(1.0, abs(brute)), (s_, k, w)
                assert accept[s_, k, w] == (ratios[s_, k, w] ** 2 > unif[s_, k, w])
                if accept[s_, k, w]:
                    pu, pd = tu, td
                    tele += np.log(abs(ratios[s_, k, w]))
        s1, l1 = np.linalg.slogdet(full_matrix(w, pu, pd))
        assert np.array_equal(pu, up["pos"][w]) and np.array_equal(pd, dn["pos"][w])
        assert abs((up["logdet"][w] + dn["logdet"][w]) - l1) < 1e-8 and up["sign"][w] * dn["sign"][w] == int(s1)
        assert abs(tele - (l1 - l0)) < 1e-8
