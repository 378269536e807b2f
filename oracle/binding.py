"""ctypes binding of oracle/qmc_oracle.c (TEST INFRASTRUCTURE; numpy in, numpy out).

Argument marshalling only: every number comes out of the C file.  See the header of
qmc_oracle.c for the passages of PAPER.md each function follows.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qmc_oracle.c")
_SRC_J = os.path.join(_HERE, "qmc_jastrow_oracle.c")
_LIB = os.path.join(_HERE, "libqmc_oracle.so")
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_fp = ctypes.POINTER(ctypes.c_float)
_ip = ctypes.POINTER(ctypes.c_int)
_bp = ctypes.POINTER(ctypes.c_ubyte)


class SweepOpts(ctypes.Structure):
    """orc_sweep_opts of qmc_oracle.c."""
    _fields_ = [("tau", ctypes.c_double), ("rprop_in", _dp), ("rprop_out", _dp), ("fcur_out", _dp),
                ("logt_out", _dp), ("b32", ctypes.c_int), ("jas", ctypes.c_void_p), ("other", _dp),
                ("nother", ctypes.c_int), ("jratio_out", _dp)]


class JastrowC(ctypes.Structure):
    """orc_jastrow of qmc_jastrow_oracle.c."""
    _fields_ = [("nfunc", ctypes.c_int), ("rc", _dp), ("M", _ip), ("poff", _ip), ("p", _dp),
                ("f_same", ctypes.c_int), ("f_opp", ctypes.c_int), ("lattice", _dp), ("nion", ctypes.c_int),
                ("ion", _dp), ("ion_func", _ip), ("range", ctypes.c_int)]


class Jastrow:
    """One- and two-body B-spline Jastrow factor (eq. 30-33) for the oracle: function table
    funcs = [(rc, p[0..M]), ...]; f_same / f_opp index the electron-electron functions (-1: none);
    ions [nion][3] with ion_func [nion]; lattice 3x3 or None (open boundary conditions)."""

    def __init__(self, funcs, f_same=-1, f_opp=-1, lattice=None, ions=None, ion_func=None, image_range=1):
        self.rc = np.ascontiguousarray([f[0] for f in funcs], dtype=np.float64)
        self.M = np.ascontiguousarray([len(f[1]) - 1 for f in funcs], dtype=np.int32)
        self.poff = np.ascontiguousarray(np.concatenate([[0], np.cumsum(self.M + 1)[:-1]]), dtype=np.int32)
        self.p = np.ascontiguousarray(np.concatenate([np.asarray(f[1], dtype=np.float64) for f in funcs]))
        self.lattice = None if lattice is None else _c64(lattice).reshape(9).copy()
        self.ions = np.zeros((0, 3)) if ions is None else _c64(ions).reshape(-1, 3).copy()
        self.ion_func = (np.zeros(0, dtype=np.int32) if ion_func is None
                         else np.ascontiguousarray(ion_func, dtype=np.int32))
        assert len(self.ion_func) == len(self.ions)
        self.c = JastrowC(len(funcs), _d(self.rc), self.M.ctypes.data_as(_ip), self.poff.ctypes.data_as(_ip),
                          _d(self.p), int(f_same), int(f_opp), _d(self.lattice), len(self.ions), _d(self.ions),
                          self.ion_func.ctypes.data_as(_ip), int(image_range))

    def ref(self):
        return ctypes.cast(ctypes.pointer(self.c), ctypes.c_void_p)


def build(force=False):
    """Compile qmc_oracle.c with gcc -O2 (no fast-math, no intrinsics) into oracle/."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_J))):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, _SRC_J, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        lib.orc_spline_vgl.restype = ctypes.c_int
        lib.orc_spline_vgl.argtypes = [ctypes.c_int] * 4 + [_dp, _fp, ctypes.c_int, _dp, _dp, _dp, _dp]
        lib.orc_spline_vgl_twist.restype = ctypes.c_int
        lib.orc_spline_vgl_twist.argtypes = ([ctypes.c_int] * 4 + [_dp, _fp, ctypes.c_int, _dp, _ip,
                                             _dp, _dp, _dp])
        lib.orc_lu_inverse.restype = ctypes.c_int
        lib.orc_lu_inverse.argtypes = [ctypes.c_int, _dp, _dp, _dp, _ip]
        lib.orc_binv_from_A.restype = ctypes.c_int
        lib.orc_binv_from_A.argtypes = [ctypes.c_int, _dp, _dp, _dp, _ip]
        lib.orc_det_ratio.restype = ctypes.c_double
        lib.orc_det_ratio.argtypes = [ctypes.c_int, _dp, ctypes.c_int, _dp]
        lib.orc_sm_update.restype = ctypes.c_int
        lib.orc_sm_update.argtypes = [ctypes.c_int, _dp, ctypes.c_int, _dp, ctypes.c_double]
        lib.orc_slater_matrix.restype = ctypes.c_int
        lib.orc_slater_matrix.argtypes = [ctypes.c_int] * 4 + [_dp, _fp, ctypes.c_int, ctypes.c_int, _dp, _dp]
        lib.orc_sweep.restype = ctypes.c_int
        lib.orc_sweep.argtypes = ([ctypes.c_int] * 4 + [_dp, _fp, ctypes.c_int, ctypes.c_int,
                                  _dp, _dp, _dp, _dp, _ip, _dp, _dp, ctypes.c_int, ctypes.c_int,
                                  _dp, _bp, _bp, _fp, _dp, ctypes.c_int, ctypes.c_int, _dp,
                                  ctypes.c_int, _dp])
        lib.orc_sweep_ex.restype = ctypes.c_int
        lib.orc_sweep_ex.argtypes = lib.orc_sweep.argtypes + [ctypes.POINTER(SweepOpts)]
        lib.orc_init_walkers.restype = ctypes.c_int
        lib.orc_init_walkers.argtypes = ([ctypes.c_int] * 4 + [_dp, _fp, ctypes.c_int, ctypes.c_int,
                                         _dp, _dp, _dp, _dp, _ip, ctypes.c_int])
        lib.orc_det_kinetic.restype = ctypes.c_int
        lib.orc_det_kinetic.argtypes = ([ctypes.c_int] * 4 + [_dp, _fp, ctypes.c_int, ctypes.c_int] + [_dp] * 6)
        lib.orc_max_threads.restype = ctypes.c_int
        lib.orc_max_threads.argtypes = []
        lib.orc_b3.restype = ctypes.c_double
        lib.orc_b3.argtypes = [ctypes.c_double]
        lib.orc_jastrow_u.restype = ctypes.c_double
        lib.orc_jastrow_u.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int, _dp]
        lib.orc_min_image.restype = ctypes.c_double
        lib.orc_min_image.argtypes = [_dp, _dp, _dp, ctypes.c_int]
        lib.orc_jastrow_value.restype = ctypes.c_double
        lib.orc_jastrow_value.argtypes = [ctypes.c_void_p, ctypes.c_int, _dp, ctypes.c_int, _dp]
        lib.orc_jastrow_dj.restype = ctypes.c_double
        lib.orc_jastrow_dj.argtypes = [ctypes.c_void_p, ctypes.c_int, _dp, ctypes.c_int, _dp, ctypes.c_int, _dp]
        _lib = lib
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _c64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _coefs(coefs):
    assert coefs.dtype == np.float32 and coefs.ndim == 4 and coefs.flags.c_contiguous
    return coefs


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def max_threads():
    return int(_load().orc_max_threads())


def spline_vgl(coefs, lattice, pos, want_gl=True):
    """coefs float32 [nx][ny][nz][norb]; pos [npos][3] -> v [npos][norb], g [npos][3][norb], l."""
    lib = _load()
    coefs = _coefs(coefs)
    nx, ny, nz, norb = coefs.shape
    lat = _c64(lattice).reshape(9)
    pos = _c64(pos).reshape(-1, 3)
    npos = pos.shape[0]
    v = np.empty((npos, norb))
    g = np.empty((npos, 3, norb)) if want_gl else None
    l = np.empty((npos, norb)) if want_gl else None
    rc = lib.orc_spline_vgl(nx, ny, nz, norb, _d(lat), coefs.ctypes.data_as(_fp), npos,
                            _d(pos), _d(v), _d(g), _d(l))
    _check(rc, "spline_vgl")
    return (v, g, l) if want_gl else v


def spline_vgl_twist(coefs, lattice, pos, half_twist):
    """spline_vgl for real orbitals at a half twist: half_twist = 3 flags, 1 = twist angle pi
    along that cell vector (eq. 43)."""
    lib = _load()
    coefs = _coefs(coefs)
    nx, ny, nz, norb = coefs.shape
    lat = _c64(lattice).reshape(9)
    pos = _c64(pos).reshape(-1, 3)
    npos = pos.shape[0]
    tw = np.ascontiguousarray(np.asarray(half_twist, dtype=np.int32).reshape(3))
    v = np.empty((npos, norb))
    g = np.empty((npos, 3, norb))
    l = np.empty((npos, norb))
    rc = lib.orc_spline_vgl_twist(nx, ny, nz, norb, _d(lat), coefs.ctypes.data_as(_fp), npos,
                                  _d(pos), tw.ctypes.data_as(_ip), _d(v), _d(g), _d(l))
    _check(rc, "spline_vgl_twist")
    return v, g, l


def lu_inverse(A):
    """A [n][n] -> (Ainv, log|det A|, sign)."""
    lib = _load()
    A = _c64(A)
    n = A.shape[0]
    Ainv = np.empty((n, n))
    ld = ctypes.c_double(0.0)
    sg = ctypes.c_int(0)
    rc = lib.orc_lu_inverse(n, _d(A), _d(Ainv), ctypes.byref(ld), ctypes.byref(sg))
    _check(rc, "lu_inverse")
    return Ainv, ld.value, sg.value


def binv_from_A(A):
    """A [n][n] -> (B = (A^-1)^T, log|det A|, sign)."""
    lib = _load()
    A = _c64(A)
    n = A.shape[0]
    B = np.empty((n, n))
    ld = ctypes.c_double(0.0)
    sg = ctypes.c_int(0)
    rc = lib.orc_binv_from_A(n, _d(A), _d(B), ctypes.byref(ld), ctypes.byref(sg))
    _check(rc, "binv_from_A")
    return B, ld.value, sg.value


def det_ratio(B, k, phi):
    lib = _load()
    B = _c64(B)
    phi = _c64(phi)
    return float(lib.orc_det_ratio(B.shape[0], _d(B), int(k), _d(phi)))


def sm_update(B, k, phi, R):
    """Returns the updated copy of B."""
    lib = _load()
    B = _c64(B).copy()
    phi = _c64(phi)
    _check(lib.orc_sm_update(B.shape[0], _d(B), int(k), _d(phi), float(R)), "sm_update")
    return B


def slater_matrix(coefs, lattice, pos):
    """pos [nw][nel][3] -> A [nw][nel][nel], A[w][i][j] = phi_j(r_wi)."""
    lib = _load()
    coefs = _coefs(coefs)
    nx, ny, nz, norb = coefs.shape
    lat = _c64(lattice).reshape(9)
    pos = _c64(pos)
    nw, nel, _ = pos.shape
    A = np.empty((nw, nel, nel))
    rc = lib.orc_slater_matrix(nx, ny, nz, norb, _d(lat), coefs.ctypes.data_as(_fp), nw, nel,
                               _d(pos), _d(A))
    _check(rc, "slater_matrix")
    return A


def det_kinetic(coefs, lattice, pos, B):
    """Kinetic term of the local energy of Psi = det A (eq. 3, eq. 37): returns a dict with
    grad [nw][nel][3] = grad_i det / det, lap [nw][nel] = lap_i det / det, one [nw][nel] (= 1 when B
    is the transposed inverse at pos) and ekin [nw] = -1/2 sum_i lap."""
    lib = _load()
    coefs = _coefs(coefs)
    nx, ny, nz, norb = coefs.shape
    lat = _c64(lattice).reshape(9)
    pos = _c64(pos)
    nw, nel, _ = pos.shape
    B = _c64(B, (nw, nel, nel))
    grad, lap, one, ekin = np.empty((nw, nel, 3)), np.empty((nw, nel)), np.empty((nw, nel)), np.empty(nw)
    rc = lib.orc_det_kinetic(nx, ny, nz, norb, _d(lat), coefs.ctypes.data_as(_fp), nw, nel, _d(pos), _d(B),
                             _d(grad), _d(lap), _d(one), _d(ekin))
    _check(rc, "det_kinetic")
    return dict(grad=grad, lap=lap, one=one, ekin=ekin)


def init_walkers(coefs, lattice, pos, nthreads=1, want_A=False):
    """pos [nw][nel][3] -> (B [nw][nel][nel], logdet [nw], sign [nw]) (+ A if want_A)."""
    lib = _load()
    coefs = _coefs(coefs)
    nx, ny, nz, norb = coefs.shape
    lat = _c64(lattice).reshape(9)
    pos = _c64(pos)
    nw, nel, _ = pos.shape
    A = np.empty((nw, nel, nel)) if want_A else None
    B = np.empty((nw, nel, nel))
    ld = np.empty(nw)
    sg = np.empty(nw, dtype=np.int32)
    rc = lib.orc_init_walkers(nx, ny, nz, norb, _d(lat), coefs.ctypes.data_as(_fp), nw, nel, _d(pos),
                              _d(A), _d(B), _d(ld), sg.ctypes.data_as(_ip), int(nthreads))
    _check(rc, "init_walkers")
    return (B, ld, sg, A) if want_A else (B, ld, sg)


def sweep(coefs, lattice, pos, B, logdet, sign, delta, unif, A=None, iel_count=None,
          forced=None, phi_in=None, want_phi=False, mode=0, nthreads=1, want_bnorm=False,
          fixed_node=False, want_force=False, tau=0.0, rprop_in=None, b32=0, jastrow=None, other=None):
    """Run nsweeps particle-by-particle sweeps.  Inputs are copied; returns a dict with
    pos, B, A, logdet, sign, ratios [nsweeps][nel][nw], accept (uint8, same shape), phi, force
    (F = 2 grad log|Psi| of the moved electron at the proposed configuration, [nsweeps][nel][nw][3]).
    tau > 0: drift moves (delta = the Gaussian part chi ~ N(0, tau)); adds rprop, fcur, logt to the
    result; rprop_in replays given proposals.  b32: fp32-stored inverse (1 = rounded after every
    accepted update, K >= 2 = at the end of every window of K steps); B must hold fp32 values."""
    lib = _load()
    coefs = _coefs(coefs)
    nx, ny, nz, norb = coefs.shape
    lat = _c64(lattice).reshape(9)
    pos = _c64(pos).copy()
    nw, nel, _ = pos.shape
    B = _c64(B, (nw, nel, nel)).copy()
    A = None if A is None else _c64(A, (nw, nel, nel)).copy()
    logdet = _c64(logdet, (nw,)).copy()
    sign = np.ascontiguousarray(sign, dtype=np.int32).copy()
    delta = _c64(delta)
    nsweeps = delta.shape[0]
    assert delta.shape == (nsweeps, nel, nw, 3)
    unif = _c64(unif, (nsweeps, nel, nw))
    if iel_count is None:
        iel_count = nel
    ratios = np.zeros((nsweeps, nel, nw))
    accept = np.zeros((nsweeps, nel, nw), dtype=np.uint8)
    f_ptr = None
    if forced is not None:
        forced = np.ascontiguousarray(forced, dtype=np.uint8)
        assert forced.shape == (nsweeps, nel, nw)
        f_ptr = forced.ctypes.data_as(_bp)
    p_ptr = None
    if phi_in is not None:
        assert phi_in.dtype == np.float32 and phi_in.flags.c_contiguous
        assert phi_in.shape == (nsweeps, nel, nw, nel)
        p_ptr = phi_in.ctypes.data_as(_fp)
    phi_out = np.zeros((nsweeps, nel, nw, nel)) if want_phi else None
    bnorm = np.zeros((nsweeps, nel, nw)) if want_bnorm else None
    force = np.zeros((nsweeps, nel, nw, 3)) if want_force else None
    drift = tau > 0.0
    rprop = np.zeros((nsweeps, nel, nw, 3)) if drift else None
    fcur = np.zeros((nsweeps, nel, nw, 3)) if drift else None
    logt = np.zeros((nsweeps, nel, nw)) if drift else None
    if rprop_in is not None:
        rprop_in = _c64(rprop_in, (nsweeps, nel, nw, 3))
    if b32:
        assert np.array_equal(B, B.astype(np.float32).astype(np.float64)), "b32: B must hold fp32 values"
    jratio = None
    nother = 0
    if jastrow is not None:
        jratio = np.ones((nsweeps, nel, nw))
        if other is not None:
            other = _c64(other)
            assert other.shape[0] == nw and other.shape[2] == 3
            nother = other.shape[1]
    opts = SweepOpts(float(tau), _d(rprop_in), _d(rprop), _d(fcur), _d(logt), int(b32),
                     None if jastrow is None else jastrow.ref(), _d(other) if nother else None, nother, _d(jratio))
    rc = lib.orc_sweep_ex(nx, ny, nz, norb, _d(lat), coefs.ctypes.data_as(_fp), nw, nel,
                          _d(pos), _d(B), _d(A), _d(logdet), sign.ctypes.data_as(_ip),
                          _d(delta), _d(unif), nsweeps, int(iel_count), _d(ratios),
                          accept.ctypes.data_as(_bp), f_ptr, p_ptr, _d(phi_out), int(mode),
                          int(nthreads), _d(bnorm), int(bool(fixed_node)), _d(force), ctypes.byref(opts))
    _check(rc, "sweep")
    return dict(pos=pos, B=B, A=A, logdet=logdet, sign=sign, ratios=ratios, accept=accept,
                phi=phi_out, bnorm=bnorm, force=force, rprop=rprop, fcur=fcur, logt=logt, jratio=jratio)


def b3(x):
    """Cardinal cubic B-spline of eq. 33 (support [-3, 1), centred at -1)."""
    return float(_load().orc_b3(float(x)))


def jastrow_u(r, rc, p):
    """u(r) of eq. 33 with control points p[0..M] and cutoff rc."""
    p = _c64(p)
    return float(_load().orc_jastrow_u(float(r), float(rc), len(p) - 1, _d(p)))


def min_image(lattice, a, b, image_range=1):
    lat = None if lattice is None else _c64(lattice).reshape(9)
    return float(_load().orc_min_image(_d(lat), _d(_c64(a, (3,))), _d(_c64(b, (3,))), int(image_range)))


def jastrow_value(jas, pos, other=None):
    """J (eq. 30, one- and two-body terms) of ONE walker: pos [nel][3], other [nother][3] (other spin)."""
    pos = _c64(pos).reshape(-1, 3)
    other = np.zeros((0, 3)) if other is None else _c64(other).reshape(-1, 3)
    return float(_load().orc_jastrow_value(jas.ref(), len(pos), _d(pos), len(other), _d(other) if len(other) else None))


def jastrow_dj(jas, pos, k, rnew, other=None):
    """J(electron k at rnew) - J(electron k at pos[k]) of ONE walker; the move's ratio is exp(-dJ)."""
    pos = _c64(pos).reshape(-1, 3)
    other = np.zeros((0, 3)) if other is None else _c64(other).reshape(-1, 3)
    return float(_load().orc_jastrow_dj(jas.ref(), len(pos), _d(pos), len(other), _d(other) if len(other) else None,
                                        int(k), _d(_c64(rnew, (3,)))))


def wf_sweep(spin, delta, unif, forced=None, phi_in=None, nthreads=1, **kw):
    """Psi_T = D_up D_dn (eq. 26 with one determinant per spin, no Jastrow): a sweep iterates over
    the up electrons, then the down electrons (L195); moving an up electron leaves D_dn unchanged, so the
    sweep IS the up sweep followed by the down sweep.  Marshalling only: the arrays are sliced per spin and
    `sweep` is called once per spin and sweep.

    spin: two dicts (up, down) with coefs, lattice, pos, B, logdet, sign.  delta [nsweeps][nup+ndn][nw][3],
    unif / forced [nsweeps][nup+ndn][nw]; phi_in: None or a pair of float32 [nsweeps][n_s][nw][n_s].
    With jastrow=...: the electrons of the other spin, at their current positions, are the fixed `other`
    particles of each per-spin sweep (opposite-spin function).
    Returns (up result, down result, ratios [nsweeps][nup+ndn][nw], accept likewise)."""
    nup, ndn = spin[0]["pos"].shape[1], spin[1]["pos"].shape[1]
    nsweeps, n, nw, _ = delta.shape
    assert n == nup + ndn
    state = [dict(pos=s_["pos"], B=s_["B"], logdet=s_["logdet"], sign=s_["sign"]) for s_ in spin]
    ratios = np.zeros((nsweeps, n, nw))
    accept = np.zeros((nsweeps, n, nw), dtype=np.uint8)
    out = [None, None]
    for sw in range(nsweeps):
        for sp, (lo, hi) in enumerate(((0, nup), (nup, n))):
            st = state[sp]
            r = sweep(spin[sp]["coefs"], spin[sp]["lattice"], st["pos"], st["B"], st["logdet"], st["sign"],
                      np.ascontiguousarray(delta[sw:sw + 1, lo:hi]), np.ascontiguousarray(unif[sw:sw + 1, lo:hi]),
                      forced=None if forced is None else np.ascontiguousarray(forced[sw:sw + 1, lo:hi]),
                      phi_in=None if phi_in is None else np.ascontiguousarray(phi_in[sp][sw:sw + 1]),
                      nthreads=nthreads, other=state[1 - sp]["pos"] if kw.get("jastrow") is not None else None, **kw)
            state[sp] = dict(pos=r["pos"], B=r["B"], logdet=r["logdet"], sign=r["sign"])
            ratios[sw, lo:hi] = r["ratios"][0]
            accept[sw, lo:hi] = r["accept"][0]
            out[sp] = r
    return out[0], out[1], ratios, accept
