"""Pins of the oracle's half-twist spline evaluation (oracle.spline_vgl_twist; PAPER.md L449-455
sec 9.2, eq. 43 with twist angle pi; reading R:A23 in DESIGN.md) -- none re-types its sign rule:

  T-a  Bloch condition, eq. 43: phi(r + L_d) = -phi(r) along twisted cell vectors, +phi(r) along
       the others; gradient and Laplacian likewise
  T-b  the antiperiodic table of n points is one half of a PERIODIC table of 2n points with
       c[i + n] = -c[i] on a cell twice as long: the (scipy-pinned) periodic evaluator on the
       doubled table gives the same value, gradient and Laplacian, inside and outside the cell
  T-c  scipy.interpolate.BSpline tensor product over the sign-extended control points
  T-d  no twist = oracle.spline_vgl, bit for bit
  T-e  an antiperiodic plane wave cos(pi (2 k + 1) u) sampled into the table is reproduced at the
       grid nodes up to the B-spline filter factor, across the twisted wrap
  T-f  C2 continuity across the twisted cell face
"""
import itertools

import numpy as np
import pytest
from scipy.interpolate import BSpline

import oracle

SKEW = np.array([[3.1, 0.2, -0.1], [0.4, 2.7, 0.3], [-0.2, 0.5, 3.4]])
ORTHO = np.diag([2.4, 3.0, 3.5])
TWISTS = [t for t in itertools.product((0, 1), repeat=3) if any(t)]


def rand_table(rng, grid, norb):
    return rng.uniform(-1, 1, size=(*grid, norb)).astype(np.float32)


# ----------------------------------------------------------------------------- T-a
@pytest.mark.parametrize("tw", TWISTS)
def test_bloch_condition(tw):
    rng = np.random.default_rng(11)
    grid, norb = (6, 5, 7), 4
    coefs = rand_table(rng, grid, norb)
    pos = rng.uniform(-1.5, 1.5, size=(25, 3)) @ SKEW
    v0, g0, l0 = oracle.spline_vgl_twist(coefs, SKEW, pos, tw)
    assert np.max(np.abs(v0)) > 0.1
    for m in ([1, 0, 0], [0, 1, 0], [0, 0, 1], [1, -2, 3], [-3, 1, 1], [2, 2, -4]):
        sign = (-1.0) ** sum(mi * ti for mi, ti in zip(m, tw))
        v1, g1, l1 = oracle.spline_vgl_twist(coefs, SKEW, pos + np.asarray(m, dtype=float) @ SKEW, tw)
        assert np.max(np.abs(v1 - sign * v0)) < 1e-12
        assert np.max(np.abs(g1 - sign * g0)) < 1e-10
        assert np.max(np.abs(l1 - sign * l0)) < 1e-8


# ----------------------------------------------------------------------------- T-b
@pytest.mark.parametrize("lat", [ORTHO, SKEW])
@pytest.mark.parametrize("tw", TWISTS)
def test_doubled_periodic_table(lat, tw):
    rng = np.random.default_rng(12)
    grid, norb = (5, 4, 6), 3
    coefs = rand_table(rng, grid, norb)
    big, lat2 = coefs, lat.copy()
    for d in range(3):
        if tw[d]:
            big = np.concatenate([big, -big], axis=d)
            lat2[d] = 2.0 * lat2[d]
    pos = rng.uniform(-2.2, 2.2, size=(120, 3)) @ lat
    v, g, l = oracle.spline_vgl_twist(coefs, lat, pos, tw)
    v2, g2, l2 = oracle.spline_vgl(np.ascontiguousarray(big), lat2, pos)
    assert np.max(np.abs(v - v2)) < 1e-13
    assert np.max(np.abs(g - g2)) < 1e-12
    assert np.max(np.abs(l - l2)) < 1e-11


# ----------------------------------------------------------------------------- T-c
def _scipy_basis(n, s, nu):
    """Uniform cubic B-spline basis, control point m supported on [m-3, m+1) (knots j - 3)."""
    ncoef = n + 3
    t = np.arange(-3, ncoef + 1, dtype=np.float64)
    return BSpline(t, np.eye(ncoef), 3)(s, nu=nu)


@pytest.mark.parametrize("tw", [(1, 0, 0), (0, 1, 1), (1, 1, 1)])
def test_against_scipy_sign_extended(tw):
    rng = np.random.default_rng(13)
    lat, grid, norb = SKEW, (6, 5, 7), 4
    coefs = rand_table(rng, grid, norb)
    pos = rng.uniform(-1, 2, size=(60, 3)) @ lat
    li = np.linalg.inv(lat)
    u = pos @ li
    img = np.floor(u)
    s = (u - img) * np.asarray(grid, dtype=np.float64)
    J = li * np.asarray(grid, dtype=np.float64)[None, :]
    ext = coefs.astype(np.float64)
    for d in range(3):
        head = np.take(ext, range(3), axis=d)
        ext = np.concatenate([ext, -head if tw[d] else head], axis=d)   # control points n..n+2
    phase = (-1.0) ** (img @ np.asarray(tw, dtype=np.float64))          # image of the point itself
    Bs = [[_scipy_basis(grid[d], s[:, d], nu) for nu in range(3)] for d in range(3)]

    def contract(a, b, c):
        return phase[:, None] * np.einsum("pi,pj,pk,ijkn->pn", Bs[0][a], Bs[1][b], Bs[2][c], ext)

    v_ref = contract(0, 0, 0)
    d1 = np.stack([contract(1, 0, 0), contract(0, 1, 0), contract(0, 0, 1)], axis=1)
    H = np.empty((len(pos), 3, 3, norb))
    orders = {(0, 0): (2, 0, 0), (1, 1): (0, 2, 0), (2, 2): (0, 0, 2),
              (0, 1): (1, 1, 0), (0, 2): (1, 0, 1), (1, 2): (0, 1, 1)}
    for (d, e), o in orders.items():
        H[:, d, e] = H[:, e, d] = contract(*o)
    g_ref = np.einsum("jd,pdn->pjn", J, d1)
    l_ref = np.einsum("jd,je,pden->pn", J, J, H)
    v, g, l = oracle.spline_vgl_twist(coefs, lat, pos, tw)
    assert np.max(np.abs(v - v_ref)) < 1e-13
    assert np.max(np.abs(g - g_ref)) < 1e-12
    assert np.max(np.abs(l - l_ref)) < 1e-11


# ----------------------------------------------------------------------------- T-d
def test_no_twist_is_the_periodic_evaluator():
    rng = np.random.default_rng(14)
    coefs = rand_table(rng, (5, 6, 4), 5)
    pos = rng.uniform(-2, 2, size=(40, 3)) @ SKEW
    a = oracle.spline_vgl(coefs, SKEW, pos)
    b = oracle.spline_vgl_twist(coefs, SKEW, pos, (0, 0, 0))
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


# ----------------------------------------------------------------------------- T-e
def test_antiperiodic_plane_wave_at_nodes():
    """c[i] = cos(pi (2k+1) i / n + ph): at node s = j the cubic B-spline gives
    (c[j-... ]) -> (1/6)(c[j] + 4 c[j+1] + c[j+2]) = cos(theta (j+1) + ph) (2 + cos theta) / 3,
    theta = pi (2k+1) / n, for EVERY integer j only if the wrap carries the factor -1."""
    n, k, ph = 12, 2, 0.3
    theta = np.pi * (2 * k + 1) / n
    i = np.arange(n)
    coefs = np.zeros((n, 1, 1, 1), dtype=np.float64)
    coefs[:, 0, 0, 0] = np.cos(theta * i + ph)
    coefs32 = coefs.astype(np.float32)
    c = coefs32[:, 0, 0, 0].astype(np.float64)
    L = 2.0
    lat = np.diag([L, 1.0, 1.0])
    j = np.arange(-2 * n, 3 * n)                      # nodes in five images of the cell
    pos = np.zeros((len(j), 3))
    pos[:, 0] = j * (L / n)
    v, g, l = oracle.spline_vgl_twist(coefs32, lat, pos, (1, 0, 0))
    # the table as rounded to fp32, extended antiperiodically by hand
    cext = lambda q: (-1.0) ** (q // n) * c[q % n]
    ref = np.array([(cext(q) + 4 * cext(q + 1) + cext(q + 2)) / 6.0 for q in j])
    assert np.max(np.abs(v[:, 0] - ref)) < 1e-14
    closed = np.cos(theta * (j + 1) + ph) * (2 + np.cos(theta)) / 3.0
    assert np.max(np.abs(v[:, 0] - closed)) < 5e-7      # fp32 rounding of the table only
    # and the periodic evaluator does NOT reproduce it across the wrap
    vp = oracle.spline_vgl(coefs32, lat, pos, want_gl=False)
    assert np.max(np.abs(vp[:, 0] - closed)) > 0.1


# ----------------------------------------------------------------------------- T-f
def test_c2_across_the_twisted_face():
    rng = np.random.default_rng(15)
    grid, norb, lat, tw = (6, 7, 5), 3, SKEW, (1, 0, 1)
    coefs = rand_table(rng, grid, norb)
    eps = 1e-9
    for d in range(3):
        for face in (0, grid[d]):
            u = rng.uniform(0.05, 0.95, size=3)
            u[d] = face / grid[d]
            um, up = u.copy(), u.copy()
            um[d] -= eps / grid[d]
            up[d] += eps / grid[d]
            vm, gm, lm = oracle.spline_vgl_twist(coefs, lat, (um @ lat)[None], tw)
            vp, gp, lp = oracle.spline_vgl_twist(coefs, lat, (up @ lat)[None], tw)
            assert np.max(np.abs(vm - vp)) < 1e-7
            assert np.max(np.abs(gm - gp)) < 1e-6
            assert np.max(np.abs(lm - lp)) < 1e-4
