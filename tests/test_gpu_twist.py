"""GPU parity tests of real orbitals at a half twist (qmc_spline_set_half_twist; PAPER.md L449-455
sec 9.2, eq. 43 with twist angle pi; reading R:A23) against oracle.spline_vgl_twist, through the C ABI.
Tolerances are the SPO-VGL ones of tests/parity.py (value 2e-6, gradient / Laplacian 2e-5 relative)."""
import itertools

import numpy as np
import pytest
import torch

import oracle
from paper_1802_06922_b200 import api, inputs
from tests import parity as P

pytestmark = pytest.mark.gpu

SKEW = np.array([[3.1, 0.2, -0.1], [0.4, 2.7, 0.3], [-0.2, 0.5, 3.4]]) * 2.0
TWISTS = [t for t in itertools.product((0, 1), repeat=3) if any(t)]


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    api.load_library()
    torch.cuda.set_device(0)


def ragged(nw=5, nsweeps=2, norb=37, sigma=0.25):
    return inputs.make_inputs(inputs.custom_config("ragged", (12, 10, 14), norb, SKEW, nw=nw, nsweeps=nsweeps,
                                                   sigma=sigma))


def positions(x, rng):
    """Walker electrons, images far outside the cell, cell faces and corners, the origin, and a point
    whose reduced coordinate rounds up to 1.0 (R:A7)."""
    g = np.array(x.cfg.grid)
    pos = x.pos.reshape(-1, 3)[:200]
    extra = rng.uniform(-3, 4, size=(60, 3)) @ x.lattice
    faces = (rng.integers(-2 * g, 3 * g, size=(40, 3)) / g) @ x.lattice
    tiny_neg = np.array([[-1e-18, 0.3, 0.6], [0.2, -1e-18, -1e-18]]) @ x.lattice
    return np.concatenate([pos, extra, faces, tiny_neg, np.zeros((1, 3))])


@pytest.mark.parametrize("tw", TWISTS)
def test_spo_vgl_half_twist_parity(tw):
    x = ragged()
    rng = np.random.default_rng(21)
    pos = positions(x, rng)
    vo, go, lo = oracle.spline_vgl_twist(x.coefs_numpy(), x.lattice, pos, tw)
    spline = api.Spline.create(x.coefs.to(P.dev()), x.lattice)
    v_per = api.spo_vgl(spline, P.to_dev(pos), want_gl=False)
    spline.set_half_twist(tw)
    v, g, l = api.spo_vgl(spline, P.to_dev(pos))
    P.check_vgl(v, g, l, vo, go, lo, x.cfg.norb)
    assert not torch.equal(v, v_per)                     # the twist changes the orbitals
    # eq. 43 on the device itself: a shift by cell vector d flips the sign iff d is twisted
    for d in range(3):
        v1, g1, l1 = api.spo_vgl(spline, P.to_dev(pos + x.lattice[d]))
        sgn = -1.0 if tw[d] else 1.0
        scale = float(v.abs().max())
        assert float((v1 - sgn * v).abs().max()) < 4e-6 * scale
    # back to no twist: the periodic bits again
    spline.set_half_twist((0, 0, 0))
    assert torch.equal(api.spo_vgl(spline, P.to_dev(pos), want_gl=False), v_per)
    spline.destroy()


@pytest.mark.parametrize("case", ["tiny", "small"])
def test_spo_vgl_half_twist_named_configs(case):
    x = inputs.make_inputs(case)
    rng = np.random.default_rng(22)
    pos = positions(x, rng)
    tw = (1, 0, 1)
    vo, go, lo = oracle.spline_vgl_twist(x.coefs_numpy(), x.lattice, pos, tw)
    spline = api.Spline.create(x.coefs.to(P.dev()), x.lattice)
    spline.set_half_twist(tw)
    v, g, l = api.spo_vgl(spline, P.to_dev(pos))
    P.check_vgl(v, g, l, vo, go, lo, x.cfg.norb)
    spline.destroy()


def test_half_twist_errors():
    x = inputs.make_inputs("tiny")
    spline = api.Spline.create(x.coefs.to(P.dev()), x.lattice)
    with pytest.raises(api.QmcError):
        spline.set_half_twist((0, 2, 0))
    with pytest.raises(api.QmcError):
        spline.set_half_twist((-1, 0, 0))
    spline.destroy()


@pytest.mark.parametrize("delay,accept_windows", [(0, False), (5, False), (16, True)])
def test_sweep_half_twist(delay, accept_windows):
    """A sweep on twisted orbitals: the Slater matrix and every proposal's vector come from the
    twisted evaluator (checked against the oracle's), and the determinant engine's protocol legs
    (identical-vector replay, residual with A recomputed, log-det against numpy) hold unchanged.
    sigma is large enough that electrons leave the home cell during the sweeps."""
    tw = (1, 1, 0)
    x = ragged(nw=6, nsweeps=2, norb=37, sigma=1.2)
    out = P.run_protocol(x, delay_rank=delay, free_oracle=False, accept_windows=accept_windows, half_twist=tw)
    assert 0.0 < out["accept_rate"] < 1.0
    # the vectors the sweep consumed: recorded by the GPU, recomputed by the oracle at the proposals
    spline = api.Spline.create(x.coefs.to(P.dev()), x.lattice)
    spline.set_half_twist(tw)
    pos0 = P.to_dev(x.pos)
    A_g = P.gpu_slater(spline, pos0)                                     # [nw][nel][norb] fp64 numpy
    nw, nel = x.pos.shape[0], x.cfg.norb
    vo = oracle.spline_vgl_twist(x.coefs_numpy(), x.lattice, x.pos.reshape(-1, 3), tw)[0].reshape(nw, nel, nel)
    assert np.max(np.abs(A_g - vo)) < P.TOL_V * np.max(np.abs(vo))
    det = api.Det.init(spline, pos0, delay_rank=delay, accept_windows=accept_windows)
    nsw = x.delta.shape[0]
    rec = torch.zeros((nsw, nel, nw, nel), dtype=torch.float32, device=P.dev())
    pos_g = pos0.clone()
    acc = torch.zeros(x.unif.shape, dtype=torch.uint8, device=P.dev())
    api.sweep(det, pos_g, P.to_dev(x.delta), P.to_dev(x.unif), accept_out=acc, phi_record=rec, nrecord=nw)
    torch.cuda.synchronize()
    rec, acc = rec.cpu().numpy(), acc.cpu().numpy()
    # replay the positions on the host (one fp64 add per accept) and evaluate every proposal with the oracle
    cur = x.pos.copy()
    worst, left_cell = 0.0, False
    li = np.linalg.inv(x.lattice)
    for s in range(nsw):
        for k in range(nel):
            prop = cur[:, k, :] + x.delta[s, k]                          # delta [s][k][w][3]
            u = prop @ li
            left_cell |= bool(np.any(np.floor(u) != 0))
            ref = oracle.spline_vgl_twist(x.coefs_numpy(), x.lattice, prop, tw)[0]
            worst = max(worst, float(np.max(np.abs(rec[s, k] - ref))))
            a = acc[s, k].astype(bool)
            cur[a, k, :] = prop[a]
    assert left_cell
    assert worst < P.TOL_V * np.max(np.abs(vo)), worst
    assert np.array_equal(cur, pos_g.cpu().numpy())
    det.destroy()
    spline.destroy()
