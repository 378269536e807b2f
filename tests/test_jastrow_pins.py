"""Pins of the Jastrow oracle (oracle/qmc_jastrow_oracle.c; sec 7, eq. 28-34) against facts the
paper and the mathematics fix:

  J-a  B_3 of eq. 33 = scipy's uniform cubic B-spline basis element on the knots -3..1 (de Boor recursion,
       a library routine), zero outside [-3, 1), centred at -1, partition of unity
  J-b  u(r) of eq. 33 = scipy.interpolate.BSpline with knots -3..M+1 and the control points as coefficients;
       zero at and beyond the cutoff; linear control points reproduce a straight line
  J-c  eq. 34 (cusp condition; reading R:A21): with p_0 = p_2 - 2 (r_c / M) u'(0) the slope of eq. 33 at
       r = 0 is the prescribed cusp
  J-d  minimum image: brute force over 9^3 lattice translations (numpy), skewed and orthorhombic cells,
       invariance under lattice translations of either point; open boundaries = the plain distance
  J-e  J of eq. 30: a three-particle configuration by hand; a numpy double loop with scipy's B-spline
  J-f  dJ of a single-electron move = J(R') - J(R)
  J-g  sweep with a Jastrow factor: accept <=> R^2 exp(-2 dJ) > u; the product of exp(-dJ) over the accepted
       moves telescopes to exp(-(J_final - J_initial)); a Jastrow factor of zeros changes nothing
"""
import numpy as np
import pytest
from scipy.interpolate import BSpline

import oracle
from paper_1802_06922_b200 import inputs

SKEW = np.array([[6.1, 0.4, -0.3], [0.7, 5.6, 0.5], [-0.4, 0.9, 6.4]])
ORTHO = np.diag([5.2, 6.0, 6.6])


def scipy_u(r, rc, p):
    """eq. 33 through scipy: sum_m p_m x (basis element on the knots m-3..m+1) at x = r / (rc / M)."""
    M = len(p) - 1
    x = np.atleast_1d(np.asarray(r, dtype=np.float64)) / (rc / M)
    out = np.zeros_like(x)
    for m in range(M + 1):
        elem = BSpline.basis_element(np.arange(m - 3, m + 2, dtype=np.float64), extrapolate=False)
        out += p[m] * np.nan_to_num(elem(x), nan=0.0)
    out = np.where(np.atleast_1d(np.asarray(r)) < rc, out, 0.0)
    return out if np.ndim(r) else out[0]


def brute_min_image(lat, a, b, rng_=4):
    d = np.asarray(a) - np.asarray(b)
    if lat is None:
        return float(np.linalg.norm(d))
    best = np.inf
    for i in range(-rng_, rng_ + 1):
        for j in range(-rng_, rng_ + 1):
            for k in range(-rng_, rng_ + 1):
                best = min(best, float(np.linalg.norm(d + np.array([i, j, k], dtype=np.float64) @ lat)))
    return best


# ----------------------------------------------------------------------------- J-a
def test_b3_is_the_cardinal_cubic_bspline():
    elem = BSpline.basis_element(np.array([-3.0, -2.0, -1.0, 0.0, 1.0]), extrapolate=False)
    rng = np.random.default_rng(5)
    for x in np.concatenate([rng.uniform(-3, 1, 200), [-3.0, -2.0, -1.0, 0.0, -2.5, 0.999999]]):
        assert abs(oracle.b3(x) - float(elem(x))) < 1e-15, x
    for x in [-3.0000001, -10.0, 1.0, 1.5, 7.0]:
        assert oracle.b3(x) == 0.0
    assert abs(oracle.b3(-1.0) - 2.0 / 3.0) < 1e-16 and abs(oracle.b3(-2.0) - 1.0 / 6.0) < 1e-16
    assert abs(oracle.b3(0.0) - 1.0 / 6.0) < 1e-16
    for x in rng.uniform(-1, 1, 20):          # centred at -1; partition of unity
        assert abs(oracle.b3(-1.0 + x) - oracle.b3(-1.0 - x)) < 1e-15
        assert abs(sum(oracle.b3(x - m) for m in range(-6, 7)) - 1.0) < 1e-15


# ----------------------------------------------------------------------------- J-b
@pytest.mark.parametrize("M", [1, 3, 8, 13])
def test_u_is_eq33(M):
    rng = np.random.default_rng(10 + M)
    rc = 3.7
    p = rng.uniform(-1, 1, M + 1)
    r = np.concatenate([rng.uniform(0, rc, 300), [0.0, rc * (1 - 1e-15), rc / M, 2 * rc / M]])
    got = np.array([oracle.jastrow_u(x, rc, p) for x in r])
    assert np.max(np.abs(got - scipy_u(r, rc, p))) < 1e-14
    for x in [rc, rc * 1.0000001, 10 * rc]:
        assert oracle.jastrow_u(x, rc, p) == 0.0
    # control points on a line: u(x delta) = alpha + beta (x + 1) wherever all four supporting points exist
    alpha, beta = 0.3, -0.17
    p = alpha + beta * np.arange(M + 1)
    for x in rng.uniform(0, max(M - 3, 0), 20 if M > 3 else 0):
        assert abs(oracle.jastrow_u(x * rc / M, rc, p) - (alpha + beta * (x + 1))) < 1e-13


# ----------------------------------------------------------------------------- J-c
@pytest.mark.parametrize("cusp", [-0.5, -0.25, 0.0, 0.8])
def test_cusp_condition_reading(cusp):
    """eq. 34 as printed reads p_0 = p_2 - (2M / r_c) u'(0), which is dimensionally the inverse of what
    eq. 33 implies: d/dr of eq. 33 at r = 0 is (p_2 - p_0) / (2 r_c / M).  Reading R:A21 follows eq. 33."""
    rng = np.random.default_rng(3)
    M, rc = 9, 4.2
    p = rng.uniform(-1, 1, M + 1)
    p[0] = p[2] - 2.0 * (rc / M) * cusp
    h = 1e-6
    slope = (-3 * oracle.jastrow_u(0.0, rc, p) + 4 * oracle.jastrow_u(h, rc, p) - oracle.jastrow_u(2 * h, rc, p)) / (2 * h)
    assert abs(slope - cusp) < 1e-8
    p_printed = p.copy()
    p_printed[0] = p[2] - (2.0 * M / rc) * cusp
    slope_p = (-3 * oracle.jastrow_u(0.0, rc, p_printed) + 4 * oracle.jastrow_u(h, rc, p_printed)
               - oracle.jastrow_u(2 * h, rc, p_printed)) / (2 * h)
    if cusp != 0.0:
        assert abs(slope_p - cusp) > 0.1 * abs(cusp)        # the printed form does not give the cusp


# ----------------------------------------------------------------------------- J-d
@pytest.mark.parametrize("lat", [ORTHO, SKEW, None])
def test_min_image(lat):
    rng = np.random.default_rng(8)
    for _ in range(40):
        a, b = rng.uniform(-7, 7, 3), rng.uniform(-7, 7, 3)
        got = oracle.min_image(lat, a, b)
        assert abs(got - brute_min_image(lat, a, b)) < 1e-12
        if lat is not None:
            shift = rng.integers(-3, 4, 3).astype(np.float64) @ lat
            assert abs(oracle.min_image(lat, a + shift, b) - got) < 1e-11
            assert abs(oracle.min_image(lat, a, b, image_range=2) - got) < 1e-12
        assert abs(oracle.min_image(lat, b, a) - got) < 1e-12


# ----------------------------------------------------------------------------- J-e, J-f
def make_case(lat, seed=0, nel=7, nother=5, nion=4):
    rng = np.random.default_rng(100 + seed)
    L = np.eye(3) * 6.0 if lat is None else lat
    rws = 0.5 * min(np.linalg.norm(L[0]), np.linalg.norm(L[1]), np.linalg.norm(L[2])) * 0.8
    funcs = [(rws, rng.uniform(-0.5, 0.5, 9)), (0.9 * rws, rng.uniform(-0.5, 0.5, 7)),
             (0.7 * rws, rng.uniform(-0.5, 0.5, 6)), (0.8 * rws, rng.uniform(-0.5, 0.5, 11))]
    ions = rng.uniform(0, 1, (nion, 3)) @ L
    ion_func = np.array([2 + (i % 2) for i in range(nion)], dtype=np.int32)
    jas = oracle.Jastrow(funcs, f_same=0, f_opp=1, lattice=lat, ions=ions, ion_func=ion_func)
    pos = rng.uniform(0, 1, (nel, 3)) @ L
    other = rng.uniform(0, 1, (nother, 3)) @ L
    return jas, funcs, ions, ion_func, pos, other, rng


def numpy_J(lat, funcs, ions, ion_func, pos, other):
    """eq. 30 / 31 / 32 with scipy's B-spline and the brute-force minimum image."""
    J = 0.0
    allp = [(r, 0) for r in pos] + [(r, 1) for r in other]
    for r, _ in allp:
        for R, f in zip(ions, ion_func):
            J += float(scipy_u(brute_min_image(lat, r, R), funcs[f][0], funcs[f][1]))
    for i, (ri, si) in enumerate(allp):
        for j, (rj, sj) in enumerate(allp):
            if i != j:
                f = 0 if si == sj else 1
                J += 0.5 * float(scipy_u(brute_min_image(lat, ri, rj), funcs[f][0], funcs[f][1]))
    return J


def test_jastrow_value_three_particles_by_hand():
    """One up electron, one down electron, one ion, open boundaries: J = u_I(r_1I) + u_I(r_2I) + u_opp(r_12)."""
    p_same, p_opp, p_ion = [0.3, 0.2, 0.1, 0.0], [0.5, 0.4, 0.2, 0.0], [-0.7, -0.3, -0.1, 0.0]
    jas = oracle.Jastrow([(3.0, p_same), (3.0, p_opp), (3.0, p_ion)], f_same=0, f_opp=1,
                         ions=[[0.0, 0.0, 0.0]], ion_func=[2])
    r1, r2 = np.array([1.0, 0.0, 0.0]), np.array([0.0, 2.0, 0.0])
    want = (float(scipy_u(1.0, 3.0, p_ion)) + float(scipy_u(2.0, 3.0, p_ion)) + float(scipy_u(np.sqrt(5.0), 3.0, p_opp)))
    assert abs(oracle.jastrow_value(jas, [r1], [r2]) - want) < 1e-14
    # two electrons of the SAME spin use the other function
    want_same = (float(scipy_u(1.0, 3.0, p_ion)) + float(scipy_u(2.0, 3.0, p_ion)) + float(scipy_u(np.sqrt(5.0), 3.0, p_same)))
    assert abs(oracle.jastrow_value(jas, [r1, r2]) - want_same) < 1e-14


@pytest.mark.parametrize("lat", [ORTHO, SKEW, None])
def test_jastrow_value_and_dj(lat):
    jas, funcs, ions, ion_func, pos, other, rng = make_case(lat)
    J0 = oracle.jastrow_value(jas, pos, other)
    assert abs(J0 - numpy_J(lat, funcs, ions, ion_func, pos, other)) < 1e-12
    assert abs(J0) > 1e-3
    for k in range(len(pos)):
        rnew = pos[k] + rng.normal(0, 0.8, 3)
        p2 = pos.copy()
        p2[k] = rnew
        dj = oracle.jastrow_dj(jas, pos, k, rnew, other)
        assert abs(dj - (oracle.jastrow_value(jas, p2, other) - J0)) < 1e-12
        assert abs(dj) > 1e-6
    # a move by a lattice vector changes nothing under periodic boundary conditions
    if lat is not None:
        assert abs(oracle.jastrow_dj(jas, pos, 2, pos[2] + lat[1] - 2 * lat[0], other)) < 1e-12


# ----------------------------------------------------------------------------- J-g
def test_sweep_with_jastrow():
    cfg = inputs.custom_config("jas", (10, 9, 11), 12, (5.0, 5.4, 6.1), nw=5, nsweeps=2, sigma=0.5)
    x = inputs.make_inputs(cfg)
    coefs = x.coefs_numpy()
    nw, nel = cfg.nw, cfg.norb
    jx = inputs.make_jastrow(cfg, x.lattice, nother=4)
    jas = oracle.Jastrow(jx.funcs, f_same=jx.f_same, f_opp=jx.f_opp, lattice=x.lattice, ions=jx.ions, ion_func=jx.ion_func)
    B, ld, sg = oracle.init_walkers(coefs, x.lattice, x.pos)
    plain = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif)
    out = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, jastrow=jas, other=jx.other)
    R, jr, acc, u = out["ratios"], out["jratio"], out["accept"], x.unif
    assert np.array_equal(acc.astype(bool), R * R * jr * jr > u) or np.max(np.abs(R * R * jr * jr - u)[acc.astype(bool) != (R * R * jr * jr > u)]) < 1e-12
    assert not np.array_equal(acc, plain["accept"])            # the factor matters in this case
    assert np.max(np.abs(jr - 1.0)) > 1e-2
    for w in range(nw):
        J0 = oracle.jastrow_value(jas, x.pos[w], jx.other[w])
        J1 = oracle.jastrow_value(jas, out["pos"][w], jx.other[w])
        prod = np.sum(np.log(jr[:, :, w][acc[:, :, w].astype(bool)]))
        assert abs(prod + (J1 - J0)) < 1e-10
    # exp(-dJ) of each move from orc_jastrow_dj at the positions the sweep had at that time (walker 0, sweep 0)
    pos = x.pos[0].copy()
    for k in range(nel):
        rnew = pos[k] + x.delta[0, k, 0]
        assert abs(jr[0, k, 0] - np.exp(-oracle.jastrow_dj(jas, pos, k, rnew, jx.other[0]))) < 1e-13
        if acc[0, k, 0]:
            pos[k] = rnew
    # a Jastrow factor of zeros is no Jastrow factor
    zero = oracle.Jastrow([(f[0], np.zeros_like(f[1])) for f in jx.funcs], f_same=jx.f_same, f_opp=jx.f_opp,
                          lattice=x.lattice, ions=jx.ions, ion_func=jx.ion_func)
    z = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, jastrow=zero, other=jx.other)
    assert np.array_equal(z["accept"], plain["accept"]) and np.array_equal(z["B"], plain["B"])
    # drift moves with a Jastrow factor are refused (grad J is not built)
    with pytest.raises(RuntimeError):
        oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, jastrow=jas, other=jx.other, tau=0.1)
