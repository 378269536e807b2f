"""GPU parity tests of the Jastrow factor (qmc_jastrow_*, qmc_sweep_opts_t.jastrow; eq. 28-33) against
the oracle (oracle/qmc_jastrow_oracle.c), through the C ABI.  All fp64 on both sides: the bar is rounding
(1e-12 relative to the size of the terms summed), decisions identical outside the 1e-6 band."""
import numpy as np
import pytest
import torch

import oracle
from paper_1802_06922_b200 import api, inputs
from tests import parity as P

pytestmark = pytest.mark.gpu

SKEW = np.array([[3.1, 0.2, -0.1], [0.4, 2.7, 0.3], [-0.2, 0.5, 3.4]]) * 2.0
ORTHO = np.diag([5.0, 6.0, 4.5])


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    api.load_library()
    torch.cuda.set_device(0)


def both_sides(jx, lattice):
    kw = dict(f_same=jx.f_same, f_opp=jx.f_opp, lattice=lattice, ions=jx.ions, ion_func=jx.ion_func)
    return api.Jastrow(jx.funcs, **kw), oracle.Jastrow(jx.funcs, **kw)


@pytest.mark.parametrize("lat", [ORTHO, SKEW, None], ids=["ortho", "skew", "open"])
def test_jastrow_ratio_and_value(lat):
    """qmc_jastrow_value against J of eq. 30 and qmc_jastrow_ratio against dJ of the oracle, every electron of
    every walker once; moves that leave the cell, a zero move, a move by a lattice vector."""
    L = np.eye(3) * 6.0 if lat is None else lat
    cfg = inputs.custom_config("jas", (8, 8, 8), 37, L, nw=6, nsweeps=1, sigma=0.6, index=410)
    x = inputs.make_inputs(cfg, with_table=False)
    jx = inputs.make_jastrow(cfg, L, nother=11, nion=9)
    jg, jo = both_sides(jx, lat)
    pos, other = P.to_dev(x.pos), P.to_dev(jx.other)
    nw, nel = cfg.nw, cfg.norb
    Jg = jg.value(pos, other).cpu().numpy()
    Jo = np.array([oracle.jastrow_value(jo, x.pos[w], jx.other[w]) for w in range(nw)])
    assert np.max(np.abs(Jg - Jo)) < 1e-11 * max(1.0, np.max(np.abs(Jo))), (Jg, Jo)
    Jg1 = jg.value(pos).cpu().numpy()                       # one spin only
    Jo1 = np.array([oracle.jastrow_value(jo, x.pos[w]) for w in range(nw)])
    assert np.max(np.abs(Jg1 - Jo1)) < 1e-11 * max(1.0, np.max(np.abs(Jo1)))
    worst = 0.0
    for k in range(nel):
        rnew = x.pos[:, k] + x.delta[0, k] * (8.0 if k % 5 == 0 else 1.0)       # some moves cross the cell
        if k == 3:
            rnew = x.pos[:, k].copy()                                              # zero move: dJ = 0 exactly
        if k == 4 and lat is not None:
            rnew = x.pos[:, k] + L[2] - L[0]                                       # a lattice vector: dJ = 0 to rounding
        r, dj = jg.ratio(pos, k, P.to_dev(rnew), other)
        r, dj = r.cpu().numpy(), dj.cpu().numpy()
        djo = np.array([oracle.jastrow_dj(jo, x.pos[w], k, rnew[w], jx.other[w]) for w in range(nw)])
        worst = max(worst, float(np.max(np.abs(dj - djo))))
        assert np.max(np.abs(r - np.exp(-djo))) < 1e-12 * np.max(np.exp(-djo))
        if k == 3:
            assert np.all(dj == 0.0)
        if k == 4 and lat is not None:
            assert np.max(np.abs(dj)) < 1e-12
    print("jastrow dJ max abs err", worst, "J scale", np.max(np.abs(Jo)))
    assert worst < 1e-12
    jg.destroy()


def test_jastrow_errors():
    with pytest.raises(api.QmcError):
        api.Jastrow([(1.0, [0.1])])                           # M = 0
    with pytest.raises(api.QmcError):
        api.Jastrow([(-1.0, [0.1, 0.0])])                     # r_c <= 0
    with pytest.raises(api.QmcError):
        api.Jastrow([(1.0, [0.1, 0.0])], f_same=3)            # functor index out of range
    with pytest.raises(api.QmcError):
        api.Jastrow([(1.0, [0.1, 0.0])], lattice=np.zeros((3, 3)))
    with pytest.raises(api.QmcError):
        api.Jastrow([(1.0, np.zeros(300))])                   # too many control points


def _case(name):
    if name == "ragged37_skew":
        return inputs.make_inputs(inputs.custom_config("ragged", (12, 10, 14), 37, SKEW, nw=5, nsweeps=2, sigma=0.25))
    if name == "n130":
        return inputs.make_inputs(inputs.custom_config("n130", (10, 12, 9), 130, (5.0, 6.0, 4.5), nw=3, nsweeps=1, sigma=0.2))
    return inputs.make_inputs("small", nw=16, nsweeps=1)


@pytest.mark.parametrize("case,K,aw", [("ragged37_skew", 0, False), ("ragged37_skew", 4, False), ("ragged37_skew", 16, False),
                                       ("n130", 0, False), ("n130", 7, False), ("small", 0, False), ("small", 16, False),
                                       ("small", 24, False), ("ragged37_skew", 4, True), ("n130", 7, True), ("small", 16, True)])
def test_sweep_with_jastrow(case, K, aw):
    """qmc_sweep_ex with a Jastrow factor, rank-1 and delayed handles: the oracle replays the GPU's fp32 orbital
    vectors (a) with the GPU's decisions imposed -- every determinant ratio, every exp(-dJ), positions bitwise --
    and (b) deciding for itself: decisions agree except where |R^2 exp(-2 dJ) - u| < 1e-6.  The Jastrow factor
    must matter (decisions differ from the plain sweep's)."""
    x = _case(case)
    cfg = x.cfg
    nw, nel, nsw = x.pos.shape[0], cfg.norb, x.delta.shape[0]
    jx = inputs.make_jastrow(cfg, x.lattice, nother=9, nw=nw)
    jg, jo = both_sides(jx, x.lattice)
    spline = api.Spline.create(x.coefs.to(P.dev()), x.lattice)
    pos0 = P.to_dev(x.pos)
    det = api.Det.init(spline, pos0, delay_rank=K, accept_windows=aw)      # aw: windows closed on K accepted moves
    B0 = det.get_inverse().cpu().numpy()
    ld0, sg0, _ = (t.cpu().numpy() for t in det.get_stats())
    pos = pos0.clone()
    d_t, u_t, other = P.to_dev(x.delta), P.to_dev(x.unif), P.to_dev(jx.other)
    R = torch.zeros_like(u_t)
    jr = torch.zeros_like(u_t)
    acc = torch.zeros(u_t.shape, dtype=torch.uint8, device=P.dev())
    rec = torch.zeros((nsw, nel, nw, nel), dtype=torch.float32, device=P.dev())
    api.sweep(det, pos, d_t, u_t, ratios_out=R, accept_out=acc, phi_record=rec, nrecord=nw, jastrow=jg,
              jastrow_other=other, jratio_out=jr)
    torch.cuda.synchronize()
    R, jr, acc, rec = R.cpu().numpy(), jr.cpu().numpy(), acc.cpu().numpy(), np.ascontiguousarray(rec.cpu().numpy())
    dummy = np.zeros((1, 1, 1, nel), np.float32)
    nth = oracle.max_threads()
    rep = oracle.sweep(dummy, x.lattice, x.pos, B0, ld0, sg0, x.delta, x.unif, forced=acc, phi_in=rec, jastrow=jo,
                       other=jx.other, nthreads=nth)
    assert np.max(np.abs(R - rep["ratios"]) / np.maximum(np.abs(rep["ratios"]), 1e-300)) < P.TOL_RATIO
    ej = float(np.max(np.abs(jr - rep["jratio"]) / rep["jratio"]))
    assert ej < 1e-11, ej
    assert np.array_equal(pos.cpu().numpy(), rep["pos"])
    Bg = det.get_inverse().cpu().numpy()
    assert np.max(np.abs(Bg - rep["B"])) < P.TOL_BINV * max(1.0, np.max(np.abs(rep["B"])))
    free = oracle.sweep(dummy, x.lattice, x.pos, B0, ld0, sg0, x.delta, x.unif, phi_in=rec, jastrow=jo, other=jx.other,
                        nthreads=nth)
    ndiv = 0
    for w in range(nw):
        a_g, a_o = acc.reshape(-1, nw)[:, w], free["accept"].reshape(-1, nw)[:, w]
        m = np.nonzero(a_g != a_o)[0]
        if len(m):
            ndiv += 1
            i = m[0]
            val = (free["ratios"].reshape(-1, nw)[i, w] * free["jratio"].reshape(-1, nw)[i, w]) ** 2
            assert abs(val - x.unif.reshape(-1, nw)[i, w]) < P.BAND, (w, i, val)
    plain = oracle.sweep(dummy, x.lattice, x.pos, B0, ld0, sg0, x.delta, x.unif, phi_in=rec, nthreads=nth)
    assert not np.array_equal(plain["accept"], acc)
    print(case, K, aw, "jastrow sweep: exp(-dJ) rel err", ej, "accept", acc.mean(), "plain accept", plain["accept"].mean(),
          "diverged", ndiv)
    # drift moves with a Jastrow factor are refused on both sides
    with pytest.raises(api.QmcError):
        api.sweep(det, pos, d_t, u_t, drift_tau=0.05, jastrow=jg)
    det.destroy()
    spline.destroy()
    jg.destroy()


@pytest.mark.parametrize("K", [0, 4])
def test_wavefunction_updn_with_jastrow(K):
    """Psi_T = e^{-J} D_up D_dn (eq. 26 with eq. 28): qmc_wf_sweep with a Jastrow factor, N_up = 37, N_dn = 29; the
    electrons of the other spin enter each spin's sweep at their current positions with the opposite-spin
    functor.  Against oracle.wf_sweep in fp64 from its own splines with the GPU's decisions imposed: exp(-dJ)
    to rounding (positions are bitwise the same), ratios within the end-to-end bound; J of the final
    configuration on both sides; the product of exp(-dJ) over accepted moves telescopes to exp(-(J1 - J0))."""
    cfgs = [inputs.custom_config("up", (12, 10, 14), 37, SKEW, nw=5, nsweeps=2, sigma=0.25, index=301),
            inputs.custom_config("dn", (12, 10, 14), 29, SKEW, nw=5, nsweeps=2, sigma=0.25, index=302)]
    xs = [inputs.make_inputs(c) for c in cfgs]
    nup, ndn, nw = 37, 29, 5
    jx = inputs.make_jastrow(cfgs[0], SKEW, nother=0, nion=8)
    jg, jo = both_sides(jx, SKEW)
    delta = np.concatenate([xs[0].delta, xs[1].delta], axis=1)
    unif = np.concatenate([xs[0].unif, xs[1].unif], axis=1)
    splines = [api.Spline.create(x.coefs.to(P.dev()), x.lattice) for x in xs]
    pos = [P.to_dev(x.pos) for x in xs]
    dets = [api.Det.init(splines[i], pos[i], delay_rank=K) for i in range(2)]
    wf = api.Wavefunction(dets[0], dets[1])
    J0 = jg.value(pos[0], pos[1]).cpu().numpy()
    R = torch.zeros(unif.shape, dtype=torch.float64, device=P.dev())
    jr = torch.zeros(unif.shape, dtype=torch.float64, device=P.dev())
    acc = torch.zeros(unif.shape, dtype=torch.uint8, device=P.dev())
    wf.sweep(pos[0], pos[1], P.to_dev(delta), P.to_dev(unif), ratios_out=R, accept_out=acc, jastrow=jg, jratio_out=jr)
    R, jr, acc = R.cpu().numpy(), jr.cpu().numpy(), acc.cpu().numpy()
    J1 = jg.value(pos[0], pos[1]).cpu().numpy()
    spin = []
    for x in xs:
        coefs = x.coefs_numpy()
        B, ld, sg = oracle.init_walkers(coefs, x.lattice, x.pos)
        spin.append(dict(coefs=coefs, lattice=x.lattice, pos=x.pos, B=B, logdet=ld, sign=sg))
    up, dn, Ro, ao = oracle.wf_sweep(spin, delta, unif, forced=acc, jastrow=jo, nthreads=oracle.max_threads())
    assert np.array_equal(pos[0].cpu().numpy(), up["pos"]) and np.array_equal(pos[1].cpu().numpy(), dn["pos"])
    # (wf_sweep returns the per-spin results of the LAST sweep; compare exp(-dJ) there)
    jr_o = np.concatenate([up["jratio"][0], dn["jratio"][0]], axis=0)
    assert np.max(np.abs(jr[-1] - jr_o) / jr_o) < 1e-11
    assert np.max(np.abs(R - Ro)) < 1e-3 * max(1.0, np.max(np.abs(Ro)))              # fp32 spline vs fp64 spline
    for w in range(nw):
        assert abs(J1[w] - oracle.jastrow_value(jo, up["pos"][w], dn["pos"][w])) < 1e-11 * max(1.0, abs(J1[w]))
        tel = np.sum(np.log(jr[:, :, w][acc[:, :, w].astype(bool)]))
        assert abs(tel + (J1[w] - J0[w])) < 1e-10
    wf.destroy()
    for d_ in dets:
        d_.destroy()
    for s_ in splines:
        s_.destroy()
    jg.destroy()
