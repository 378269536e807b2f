"""qmc_det_kinetic_noalloc (include/qmc_b200.h): the kinetic term with its Laplacian scratch in a static device
array, for callers that may not call cudaMalloc.  Checked against the existing path (qmc_det_kinetic) on the same
handle, on consecutive calls that share the array; collected last (file name) so that a failure here hides no
other test under `pytest -x`, and independent of what ran before it."""
import numpy as np
import pytest
import torch

from paper_1802_06922_b200 import api, inputs
from tests import parity as P

pytestmark = pytest.mark.gpu

SKEW = np.array([[3.1, 0.2, -0.1], [0.4, 2.7, 0.3], [-0.2, 0.5, 3.4]]) * 2.0
TOL = 1e-12          # fp64 rounding bar of the fp64-vs-fp64 checks in tests/ (the two paths sum in the same order)


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    api.load_library()
    torch.cuda.set_device(0)


def _handle(cfg, K):
    x = inputs.make_inputs(cfg)
    spline = api.Spline.create(x.coefs.to(P.dev()), x.lattice)
    pos = P.to_dev(x.pos)
    det = api.Det.init(spline, pos, delay_rank=K)
    return x, spline, pos, det


def _close(a, b):
    return float(torch.max(torch.abs(a - b))) <= TOL * max(1.0, float(torch.max(torch.abs(b))))


def test_kinetic_noalloc_matches_kinetic_on_consecutive_calls():
    """Two calls in a row on one handle (a sweep in between, so positions and inverse differ), then a smaller
    handle whose call finds the first one's Laplacians in the shared array, then the first again: each against
    qmc_det_kinetic.  The warmed-up call must leave the device's free memory unchanged."""
    xa, spa, posa, da = _handle(inputs.custom_config("na130", (10, 12, 9), 130, (5.0, 6.0, 4.5), nw=7, nsweeps=2, sigma=0.2), 16)
    xb, spb, posb, db = _handle(inputs.custom_config("na37", (12, 10, 14), 37, SKEW, nw=5, nsweeps=1, sigma=0.25), 0)
    da_delta, da_unif = P.to_dev(xa.delta), P.to_dev(xa.unif)
    out = torch.full((da.nw,), float("nan"), dtype=torch.float64, device=P.dev())
    outb = torch.full((db.nw,), float("nan"), dtype=torch.float64, device=P.dev())

    api.sweep(da, posa, da_delta[:1], da_unif[:1])
    da.kinetic_noalloc(posa, out)                                     # call 1 (delayed rank 16: flushes first)
    ref1 = da.kinetic(posa)["ekin"]
    assert torch.isfinite(out).all() and _close(out, ref1), (out, ref1)
    first = out.clone()

    api.sweep(da, posa, da_delta[1:], da_unif[1:])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    da.kinetic_noalloc(posa, out)                                     # call 2, straight after call 1's data
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                      # nothing was allocated on the device
    ref2 = da.kinetic(posa)["ekin"]
    assert _close(out, ref2), (out, ref2)
    assert not _close(first, ref2)                                    # the sweep did change the answer

    db.kinetic_noalloc(posb, outb)                                    # other shape, same array
    assert _close(outb, db.kinetic(posb)["ekin"])
    da.kinetic_noalloc(posa, out)
    assert _close(out, ref2)
    print("noalloc ekin", out[:3].tolist(), "bit-equal to qmc_det_kinetic:", bool(torch.equal(out, ref2)))
    for h in (da, db, spa, spb):
        h.destroy()


def test_kinetic_noalloc_limit():
    """nwalkers * nel = QMC_KINETIC_NOALLOC_MAX is served, one walker more is refused with a clear error and the
    output untouched."""
    nel = 16
    nw = api.KINETIC_NOALLOC_MAX // nel
    for n, ok in ((nw, True), (nw + 1, False)):
        x, sp, pos, det = _handle(inputs.custom_config("nalim", (16, 16, 16), nel, (1.0, 1.0, 1.0), nw=n, nsweeps=1, sigma=0.05), 0)
        out = torch.full((n,), -7.0, dtype=torch.float64, device=P.dev())
        if ok:
            det.kinetic_noalloc(pos, out)
            assert _close(out, det.kinetic(pos)["ekin"])
        else:
            with pytest.raises(api.QmcError, match="exceeds the static scratch"):
                det.kinetic_noalloc(pos, out)
            assert bool((out == -7.0).all())
            assert torch.isfinite(det.kinetic(pos)["ekin"]).all()     # the allocating path still serves it
        det.destroy()
        sp.destroy()
