"""Thin ctypes binding of libqmcb200.so (include/qmc_b200.h): argument marshalling only.

Every step of the hot path runs in the CUDA library; torch is used for device memory and
streams.  There is no CPU fallback: a missing library or a failing call raises.
Names follow the C ABI: Spline.create -> qmc_spline_create, spo_vgl -> qmc_spo_vgl, ...
"""
import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqmcb200.so")
_lib = None

QMC_MAX_DELAY = 32
_vp = ctypes.c_void_p

EXPORTS = [
    "qmc_last_error", "qmc_spline_create", "qmc_spline_destroy", "qmc_spline_info", "qmc_spo_vgl",
    "qmc_det_init", "qmc_det_destroy", "qmc_det_ratio", "qmc_det_accept_update", "qmc_det_flush",
    "qmc_sweep", "qmc_sweep_ex", "qmc_sweep_host", "qmc_det_get_inverse", "qmc_det_set_inverse",
    "qmc_det_get_stats", "qmc_det_info", "qmc_launch_count", "qmc_det_profile", "qmc_det_profile_read",
    "qmc_probe_fp64_dmma", "qmc_det_kinetic", "qmc_det_kinetic_noalloc", "qmc_det_ratio_points",
    "qmc_det_init_ex", "qmc_det_storage", "qmc_det_recompute", "qmc_det_residual",
    "qmc_wf_create", "qmc_wf_destroy", "qmc_wf_info", "qmc_wf_sweep", "qmc_wf_kinetic", "qmc_wf_get_stats",
    "qmc_jastrow_create", "qmc_jastrow_destroy", "qmc_jastrow_ratio", "qmc_jastrow_value", "qmc_probe_fp64_pipe",
    "qmc_spline_set_half_twist",
]
QMC_DET_FP32_INVERSE = 1
QMC_DET_ACCEPT_WINDOWS = 2
KINETIC_NOALLOC_MAX = 1 << 19      # QMC_KINETIC_NOALLOC_MAX
PROF_KINDS = ["spo_vgl", "sm_update", "delayed_window", "delayed_accept", "delayed_flush", "ratio_rowcopy"]


class SweepOpts(ctypes.Structure):
    _fields_ = [("iel_begin", ctypes.c_int), ("iel_count", ctypes.c_int),
                ("phi_record", _vp), ("nrecord", ctypes.c_int), ("fixed_node", ctypes.c_int),
                ("force_out", _vp), ("drift_tau", ctypes.c_double), ("rprop_out", _vp), ("logt_out", _vp),
                ("fcur_out", _vp), ("jastrow", _vp), ("jastrow_other", _vp), ("jastrow_nother", ctypes.c_int),
                ("jratio_out", _vp)]


class QmcError(RuntimeError):
    pass


def load_library(path=None):
    """dlopen the CUDA library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise QmcError(f"{path} is missing: run `python -m paper_1802_06922_b200.build` "
                       "(there is no CPU fallback)")
    lib = ctypes.CDLL(path)
    i, d = ctypes.c_int, ctypes.c_double
    lib.qmc_last_error.restype = ctypes.c_char_p
    lib.qmc_last_error.argtypes = []
    lib.qmc_launch_count.restype = ctypes.c_longlong
    lib.qmc_launch_count.argtypes = []
    sigs = {
        "qmc_spline_create": [ctypes.POINTER(_vp), i, i, i, i, ctypes.POINTER(d), _vp, i, _vp],
        "qmc_spline_destroy": [_vp],
        "qmc_spline_set_half_twist": [_vp, ctypes.POINTER(i)],
        "qmc_spline_info": [_vp, ctypes.POINTER(i), ctypes.POINTER(ctypes.c_size_t)],
        "qmc_spo_vgl": [_vp, i, _vp, _vp, _vp, _vp, i, _vp],
        "qmc_det_init": [ctypes.POINTER(_vp), _vp, i, i, _vp, i, _vp],
        "qmc_det_destroy": [_vp],
        "qmc_det_ratio": [_vp, i, _vp, i, _vp, _vp],
        "qmc_det_accept_update": [_vp, i, _vp, i, _vp, _vp, _vp],
        "qmc_det_flush": [_vp, _vp],
        "qmc_sweep": [_vp, _vp, _vp, _vp, _vp, i, _vp, _vp, _vp, _vp],
        "qmc_sweep_ex": [_vp, _vp, _vp, _vp, _vp, i, _vp, _vp, _vp, ctypes.POINTER(SweepOpts), _vp],
        "qmc_sweep_host": [_vp, _vp, _vp, _vp, _vp, i, _vp, _vp, _vp],
        "qmc_det_get_inverse": [_vp, _vp, _vp],
        "qmc_det_set_inverse": [_vp, _vp, _vp, _vp, _vp],
        "qmc_det_get_stats": [_vp, _vp, _vp, _vp, _vp],
        "qmc_det_info": [_vp] + [ctypes.POINTER(i)] * 4,
        "qmc_det_profile": [_vp, i],
        "qmc_det_profile_read": [_vp, ctypes.POINTER(d), ctypes.POINTER(ctypes.c_longlong)],
        "qmc_probe_fp64_dmma": [ctypes.POINTER(d), _vp],
        "qmc_probe_fp64_pipe": [i, i, i, ctypes.POINTER(d), ctypes.POINTER(d), _vp],
        "qmc_det_kinetic": [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp],
        "qmc_det_kinetic_noalloc": [_vp, _vp, _vp, _vp, _vp],
        "qmc_det_ratio_points": [_vp, i, i, _vp, i, _vp, _vp],
        "qmc_det_init_ex": [ctypes.POINTER(_vp), _vp, i, i, _vp, i, ctypes.c_uint, _vp],
        "qmc_det_storage": [_vp, ctypes.POINTER(i)],
        "qmc_det_recompute": [_vp, _vp, _vp, _vp],
        "qmc_det_residual": [_vp, _vp, _vp, i, _vp, _vp],
        "qmc_wf_create": [ctypes.POINTER(_vp), _vp, _vp, _vp, _vp],
        "qmc_wf_destroy": [_vp],
        "qmc_wf_info": [_vp] + [ctypes.POINTER(i)] * 3,
        "qmc_wf_sweep": [_vp, _vp, _vp, _vp, _vp, i, _vp, _vp, _vp, ctypes.POINTER(SweepOpts), _vp],
        "qmc_wf_kinetic": [_vp, _vp, _vp, _vp, _vp],
        "qmc_wf_get_stats": [_vp, _vp, _vp, _vp],
        "qmc_jastrow_create": [ctypes.POINTER(_vp), ctypes.POINTER(d), i, ctypes.POINTER(d), ctypes.POINTER(i),
                               ctypes.POINTER(d), i, i, i, ctypes.POINTER(d), ctypes.POINTER(i)],
        "qmc_jastrow_destroy": [_vp],
        "qmc_jastrow_ratio": [_vp, i, i, _vp, i, _vp, i, _vp, _vp, _vp, _vp],
        "qmc_jastrow_value": [_vp, i, i, _vp, i, _vp, _vp, _vp],
    }
    for name, args in sigs.items():
        fn = getattr(lib, name)
        fn.restype = i
        fn.argtypes = args
    _lib = lib
    return lib


def _check(rc, what):
    if rc != 0:
        msg = load_library().qmc_last_error().decode(errors="replace")
        raise QmcError(f"{what} failed ({rc}): {msg}")


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return _vp(s.cuda_stream)


def _ptr(t, dtype=None, allow_none=False):
    if t is None:
        if allow_none:
            return None
        raise QmcError("tensor required")
    if dtype is not None and t.dtype != dtype:
        raise QmcError(f"expected {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise QmcError("tensor must be contiguous")
    return _vp(t.data_ptr())


def _dev(t, dtype, allow_none=False):
    if t is not None and not t.is_cuda:
        raise QmcError("device tensor required")
    return _ptr(t, dtype, allow_none)


def launch_count():
    return int(load_library().qmc_launch_count())


def probe_fp64_dmma(stream=None):
    """qmc_probe_fp64_dmma: measured fp64 tensor-core (DMMA) peak of the current device, TFLOP/s."""
    out = ctypes.c_double(0.0)
    _check(load_library().qmc_probe_fp64_dmma(ctypes.byref(out), _stream(stream)), "qmc_probe_fp64_dmma")
    return out.value


def probe_fp64_pipe(mode, warps_per_sm, chains, stream=None):
    """qmc_probe_fp64_pipe: (DMMA TFLOP/s, DFMA TFLOP/s) of the fp64 pipe under the given instruction mix."""
    a, b = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(load_library().qmc_probe_fp64_pipe(int(mode), int(warps_per_sm), int(chains), ctypes.byref(a), ctypes.byref(b),
                                              _stream(stream)), "qmc_probe_fp64_pipe")
    return a.value, b.value


class Spline:
    """qmc_spline_t: the padded fp32 coefficient table on the device."""

    def __init__(self, handle, grid, norb):
        self._h = handle
        self.grid = tuple(grid)
        self.norb = int(norb)
        rp, tb = ctypes.c_int(0), ctypes.c_size_t(0)
        _check(load_library().qmc_spline_info(self._h, ctypes.byref(rp), ctypes.byref(tb)), "qmc_spline_info")
        self.row_pitch, self.table_bytes = rp.value, tb.value

    @classmethod
    def create(cls, coefs, lattice, stream=None):
        """coefs: float32 [nx][ny][nz][norb] tensor (host or device); lattice: 3x3 (rows = cell vectors)."""
        lib = load_library()
        if coefs.dtype != torch.float32 or coefs.dim() != 4 or not coefs.is_contiguous():
            raise QmcError("coefs must be a contiguous float32 [nx][ny][nz][norb] tensor")
        nx, ny, nz, norb = coefs.shape
        lat = (ctypes.c_double * 9)(*[float(x) for x in torch.as_tensor(lattice, dtype=torch.float64).reshape(9)])
        h = _vp()
        rc = lib.qmc_spline_create(ctypes.byref(h), nx, ny, nz, norb, lat, _vp(coefs.data_ptr()),
                                   1 if coefs.is_cuda else 0, _stream(stream))
        _check(rc, "qmc_spline_create")
        if not coefs.is_cuda:
            torch.cuda.synchronize()
        return cls(h, (nx, ny, nz), norb)

    def set_half_twist(self, half_twist):
        """qmc_spline_set_half_twist: 3 flags, 1 = twist angle pi along that cell vector (eq. 43)."""
        tw = (ctypes.c_int * 3)(*[int(t) for t in half_twist])
        _check(load_library().qmc_spline_set_half_twist(self._h, tw), "qmc_spline_set_half_twist")

    def destroy(self):
        if self._h:
            _check(load_library().qmc_spline_destroy(self._h), "qmc_spline_destroy")
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def spo_vgl(spline, pos, want_gl=True, ldo=None, stream=None):
    """qmc_spo_vgl: pos double [npos][3] (device) -> v [npos][ldo], g [npos][3][ldo], l [npos][ldo] (float32)."""
    lib = load_library()
    pos = pos.reshape(-1, 3)
    npos = pos.shape[0]
    ldo = spline.row_pitch if ldo is None else int(ldo)
    v = torch.empty((npos, ldo), dtype=torch.float32, device=pos.device)
    g = torch.empty((npos, 3, ldo), dtype=torch.float32, device=pos.device) if want_gl else None
    l = torch.empty((npos, ldo), dtype=torch.float32, device=pos.device) if want_gl else None
    rc = lib.qmc_spo_vgl(spline._h, npos, _dev(pos, torch.float64), _dev(v, None), _dev(g, None, True),
                         _dev(l, None, True), ldo, _stream(stream))
    _check(rc, "qmc_spo_vgl")
    return (v, g, l) if want_gl else v


def spo_vgl_into(spline, pos, v, g, l, stream=None):
    """qmc_spo_vgl into caller-provided outputs (no allocation; for timing loops)."""
    rc = load_library().qmc_spo_vgl(spline._h, pos.shape[0], _dev(pos, torch.float64), _dev(v, torch.float32),
                                    _dev(g, torch.float32, True), _dev(l, torch.float32, True), v.shape[-1],
                                    _stream(stream))
    _check(rc, "qmc_spo_vgl")


class Det:
    """qmc_det_t: fp64 (A^-1)^T of every walker plus scratch."""

    def __init__(self, handle, spline):
        self._h = handle
        self.spline = spline
        lib = load_library()
        a, b, c, e = ctypes.c_int(), ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
        _check(lib.qmc_det_info(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c), ctypes.byref(e)),
               "qmc_det_info")
        self.nw, self.nel, self.ld, self.delay_rank = a.value, b.value, c.value, e.value
        _check(lib.qmc_det_storage(self._h, ctypes.byref(a)), "qmc_det_storage")
        self.storage_bytes = a.value            # 8: fp64 inverse, 4: fp32-stored inverse

    @classmethod
    def init(cls, spline, pos, delay_rank=0, fp32_inverse=False, accept_windows=False, stream=None):
        """qmc_det_init / qmc_det_init_ex: pos double [nw][nel][3] on the device.  accept_windows: delayed windows
        close on delay_rank ACCEPTED moves (QMC_DET_ACCEPT_WINDOWS)."""
        lib = load_library()
        nw, nel, _ = pos.shape
        h = _vp()
        flags = (QMC_DET_FP32_INVERSE if fp32_inverse else 0) | (QMC_DET_ACCEPT_WINDOWS if accept_windows else 0)
        if flags:
            rc = lib.qmc_det_init_ex(ctypes.byref(h), spline._h, nw, nel, _dev(pos, torch.float64), int(delay_rank),
                                     flags, _stream(stream))
        else:
            rc = lib.qmc_det_init(ctypes.byref(h), spline._h, nw, nel, _dev(pos, torch.float64), int(delay_rank),
                                  _stream(stream))
        _check(rc, "qmc_det_init")
        return cls(h, spline)

    def recompute(self, pos, stream=None):
        """qmc_det_recompute: inverse, log|det| and sign again from scratch at pos."""
        rc = load_library().qmc_det_recompute(self._h, self.spline._h, _dev(pos, torch.float64), _stream(stream))
        _check(rc, "qmc_det_recompute")

    def residual(self, pos, nsample=4, stream=None):
        """qmc_det_residual -> double [nw]: max |B[k] . phi(r_i) - delta_ik| over nsample electrons i, all k."""
        out = torch.empty(self.nw, dtype=torch.float64, device=pos.device)
        rc = load_library().qmc_det_residual(self._h, self.spline._h, _dev(pos, torch.float64), int(nsample),
                                             _dev(out, None), _stream(stream))
        _check(rc, "qmc_det_residual")
        return out

    def destroy(self):
        if self._h:
            _check(load_library().qmc_det_destroy(self._h), "qmc_det_destroy")
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def ratio(self, iel, phi, stream=None):
        """qmc_det_ratio: phi float32 [nw][ldo] -> ratio double [nw]."""
        out = torch.empty(self.nw, dtype=torch.float64, device=phi.device)
        rc = load_library().qmc_det_ratio(self._h, int(iel), _dev(phi, torch.float32), phi.shape[-1],
                                          _dev(out, None), _stream(stream))
        _check(rc, "qmc_det_ratio")
        return out

    def ratio_points(self, iel, phi, stream=None):
        """qmc_det_ratio_points: phi float32 [nw][npts][ldo] -> ratios double [nw][npts] (no update)."""
        npts = phi.shape[1]
        out = torch.empty((self.nw, npts), dtype=torch.float64, device=phi.device)
        rc = load_library().qmc_det_ratio_points(self._h, int(iel), int(npts), _dev(phi, torch.float32),
                                                 phi.shape[-1], _dev(out, None), _stream(stream))
        _check(rc, "qmc_det_ratio_points")
        return out

    def accept_update(self, iel, phi, ratio, accept, stream=None):
        """qmc_det_accept_update: accept uint8 [nw]."""
        rc = load_library().qmc_det_accept_update(self._h, int(iel), _dev(phi, torch.float32), phi.shape[-1],
                                                  _dev(ratio, torch.float64), _dev(accept, torch.uint8),
                                                  _stream(stream))
        _check(rc, "qmc_det_accept_update")

    def flush(self, stream=None):
        _check(load_library().qmc_det_flush(self._h, _stream(stream)), "qmc_det_flush")

    def get_inverse(self, stream=None):
        """B = (A^-1)^T as double [nw][nel][nel]."""
        dev = torch.device("cuda", torch.cuda.current_device())
        out = torch.empty((self.nw, self.nel, self.nel), dtype=torch.float64, device=dev)
        _check(load_library().qmc_det_get_inverse(self._h, _dev(out, None), _stream(stream)), "qmc_det_get_inverse")
        return out

    def set_inverse(self, binv, logdet=None, sign=None, stream=None):
        rc = load_library().qmc_det_set_inverse(self._h, _dev(binv, torch.float64),
                                                _dev(logdet, torch.float64, True),
                                                _dev(sign, torch.int32, True), _stream(stream))
        _check(rc, "qmc_det_set_inverse")

    def kinetic(self, pos, want_grad=True, stream=None):
        """qmc_det_kinetic -> dict(grad [nw][nel][3] or None, lap [nw][nel], one [nw][nel], ekin [nw])."""
        dev = torch.device("cuda", torch.cuda.current_device())
        f64 = dict(dtype=torch.float64, device=dev)
        grad = torch.empty((self.nw, self.nel, 3), **f64) if want_grad else None
        lap, one, ekin = torch.empty((self.nw, self.nel), **f64), torch.empty((self.nw, self.nel), **f64), torch.empty(self.nw, **f64)
        rc = load_library().qmc_det_kinetic(self._h, self.spline._h, _dev(pos, torch.float64), _dev(grad, None, True),
                                            _dev(lap, None), _dev(one, None), _dev(ekin, None), _stream(stream))
        _check(rc, "qmc_det_kinetic")
        return dict(grad=grad, lap=lap, one=one, ekin=ekin)

    def kinetic_noalloc(self, pos, ekin_out, stream=None):
        """qmc_det_kinetic_noalloc: E_kin [nw] into the caller's `ekin_out`; no device allocation anywhere on the
        path (the Laplacian scratch is a static device array, nw * nel <= KINETIC_NOALLOC_MAX).  Calls that
        overlap on the GPU race on that array."""
        rc = load_library().qmc_det_kinetic_noalloc(self._h, self.spline._h, _dev(pos, torch.float64),
                                                    _dev(ekin_out, torch.float64), _stream(stream))
        _check(rc, "qmc_det_kinetic_noalloc")
        return ekin_out

    def profile(self, enable=True):
        """qmc_det_profile: bracket every sweep kernel with CUDA events (and reset the recorder)."""
        _check(load_library().qmc_det_profile(self._h, 1 if enable else 0), "qmc_det_profile")

    def profile_read(self):
        """qmc_det_profile_read -> {kind: (total ms, launches)}; synchronises the recorded events."""
        n = len(PROF_KINDS)
        ms = (ctypes.c_double * n)()
        cnt = (ctypes.c_longlong * n)()
        _check(load_library().qmc_det_profile_read(self._h, ms, cnt), "qmc_det_profile_read")
        return {k: (ms[j], cnt[j]) for j, k in enumerate(PROF_KINDS)}

    def get_stats(self, stream=None):
        """(logdet double [nw], sign int32 [nw], naccept int64 [nw])."""
        dev = torch.device("cuda", torch.cuda.current_device())
        ld = torch.empty(self.nw, dtype=torch.float64, device=dev)
        sg = torch.empty(self.nw, dtype=torch.int32, device=dev)
        na = torch.empty(self.nw, dtype=torch.int64, device=dev)
        rc = load_library().qmc_det_get_stats(self._h, _dev(ld, None), _dev(sg, None), _dev(na, None),
                                              _stream(stream))
        _check(rc, "qmc_det_get_stats")
        return ld, sg, na


def sweep(det, pos, delta, unif, ratios_out=None, accept_out=None, forced_accept=None, iel_begin=0,
          iel_count=0, phi_record=None, nrecord=0, fixed_node=False, force_out=None, drift_tau=0.0,
          rprop_out=None, logt_out=None, fcur_out=None, jastrow=None, jastrow_other=None, jratio_out=None,
          stream=None):
    """qmc_sweep / qmc_sweep_ex on device tensors (pos updated in place).

    jastrow: a Jastrow handle (accept iff R^2 exp(-2 dJ) > u); jastrow_other double [nw][nother][3] or None:
    the electrons of the other spin; jratio_out double [nsweeps][nel][nw] or None: exp(-dJ) of every move.

    pos double [nw][nel][3]; delta double [nsweeps][nel][nw][3]; unif double [nsweeps][nel][nw];
    ratios_out double / accept_out uint8 / forced_accept uint8: [nsweeps][nel][nw] or None;
    phi_record float32 [nsweeps][nel][nrecord][nel] or None; fixed_node: reject moves with R < 0;
    force_out double [nsweeps][nel][nw][3] or None (F = 2 grad log|Psi| at the proposed configuration).
    drift_tau > 0: drift moves (delta = chi ~ N(0, tau)); rprop_out [nsweeps][nel][nw][3], logt_out
    [nsweeps][nel][nw], fcur_out [nsweeps][nel][nw][3]: proposals, log T'/T and F at the current configuration.
    """
    lib = load_library()
    nsweeps = delta.shape[0]
    if tuple(delta.shape) != (nsweeps, det.nel, det.nw, 3) or tuple(unif.shape) != (nsweeps, det.nel, det.nw):
        raise QmcError("delta / unif shapes do not match the determinant")
    if tuple(pos.shape) != (det.nw, det.nel, 3):
        raise QmcError("pos shape does not match the determinant")
    for t in (ratios_out, accept_out, forced_accept):
        if t is not None and tuple(t.shape) != tuple(unif.shape):
            raise QmcError("per-move arrays must be [nsweeps][nel][nw]")
    args = [det._h, det.spline._h, _dev(pos, torch.float64), _dev(delta, torch.float64),
            _dev(unif, torch.float64), nsweeps, _dev(ratios_out, torch.float64, True),
            _dev(accept_out, torch.uint8, True), _dev(forced_accept, torch.uint8, True)]
    if (iel_begin or iel_count or phi_record is not None or fixed_node or force_out is not None or drift_tau
            or jastrow is not None):
        if phi_record is not None and tuple(phi_record.shape) != (nsweeps, det.nel, nrecord, det.nel):
            raise QmcError("phi_record must be [nsweeps][nel][nrecord][nel]")
        if force_out is not None and tuple(force_out.shape) != tuple(unif.shape) + (3,):
            raise QmcError("force_out must be [nsweeps][nel][nw][3]")
        opts = SweepOpts(int(iel_begin), int(iel_count),
                         None if phi_record is None else phi_record.data_ptr(), int(nrecord),
                         1 if fixed_node else 0,
                         None if force_out is None else _dev(force_out, torch.float64).value,
                         float(drift_tau),
                         None if rprop_out is None else _dev(rprop_out, torch.float64).value,
                         None if logt_out is None else _dev(logt_out, torch.float64).value,
                         None if fcur_out is None else _dev(fcur_out, torch.float64).value,
                         None if jastrow is None else jastrow._h,
                         None if jastrow_other is None else _dev(jastrow_other, torch.float64).value,
                         0 if jastrow_other is None else int(jastrow_other.shape[1]),
                         None if jratio_out is None else _dev(jratio_out, torch.float64).value)
        rc = lib.qmc_sweep_ex(*args, ctypes.byref(opts), _stream(stream))
        _check(rc, "qmc_sweep_ex")
    else:
        _check(lib.qmc_sweep(*args, _stream(stream)), "qmc_sweep")


class SweepGraph:
    """One qmc_sweep call captured into a CUDA graph and replayed (the sequential loop over
    electrons is 2-3 small launches per electron step; on the L2-resident configs -- tiny, small -- the sweep is
    launch-bound, and a graph replays its launches without the per-launch host cost).

    The tensors passed in are the graph's static buffers: refresh `delta` / `unif` in place (copy_) between
    replays; `pos`, the handle's inverse and the outputs are updated by every replay exactly as by
    `sweep(...)`.  Run one eager `sweep` first: the library allocates its scratch and streams on first use,
    which a capture must not do.  Plumbing only: torch.cuda.CUDAGraph captures the launches the library
    enqueues on torch's current stream."""

    def __init__(self, det, pos, delta, unif, **kw):
        self.graph = torch.cuda.CUDAGraph()
        self._keep = (det, pos, delta, unif, kw)
        with torch.cuda.graph(self.graph):
            sweep(det, pos, delta, unif, **kw)

    def replay(self):
        self.graph.replay()


def sweep_host(det, pos, delta, unif, ratios_out=None, accept_out=None, stream=None):
    """qmc_sweep_host on HOST tensors (ideally pinned); synchronises.  pos is updated in place."""
    lib = load_library()
    for t in (pos, delta, unif, ratios_out, accept_out):
        if t is not None and t.is_cuda:
            raise QmcError("sweep_host takes host tensors")
    nsweeps = delta.shape[0]
    rc = lib.qmc_sweep_host(det._h, det.spline._h, _ptr(pos, torch.float64), _ptr(delta, torch.float64),
                            _ptr(unif, torch.float64), nsweeps, _ptr(ratios_out, torch.float64, True),
                            _ptr(accept_out, torch.uint8, True), _stream(stream))
    _check(rc, "qmc_sweep_host")


class Jastrow:
    """qmc_jastrow_t: one- and two-body B-spline Jastrow factor (eq. 28-33).  funcs = [(r_c, p[0..M]), ...];
    f_same / f_opp: the electron-electron functors (-1 = none); lattice 3x3 or None (open boundaries);
    ions [nion][3] with functor index ion_func [nion].  Host inputs (numpy), copied to the current device."""

    def __init__(self, funcs, f_same=-1, f_opp=-1, lattice=None, ions=None, ion_func=None):
        lib = load_library()
        d, i = ctypes.c_double, ctypes.c_int
        rc_a = np.ascontiguousarray([f[0] for f in funcs], dtype=np.float64)
        m_a = np.ascontiguousarray([len(f[1]) - 1 for f in funcs], dtype=np.int32)
        p_a = np.ascontiguousarray(np.concatenate([np.asarray(f[1], dtype=np.float64) for f in funcs]))
        lat = None if lattice is None else np.ascontiguousarray(lattice, dtype=np.float64).reshape(9)
        ions = np.zeros((0, 3)) if ions is None else np.ascontiguousarray(ions, dtype=np.float64).reshape(-1, 3)
        ifn = np.zeros(0, dtype=np.int32) if ion_func is None else np.ascontiguousarray(ion_func, dtype=np.int32)
        if len(ifn) != len(ions):
            raise QmcError("ion_func must have one entry per ion")
        dp = lambda a: None if a is None or a.size == 0 else a.ctypes.data_as(ctypes.POINTER(d))
        ip = lambda a: None if a.size == 0 else a.ctypes.data_as(ctypes.POINTER(i))
        h = _vp()
        rc = lib.qmc_jastrow_create(ctypes.byref(h), dp(lat), len(funcs), dp(rc_a), ip(m_a), dp(p_a), int(f_same),
                                    int(f_opp), len(ions), dp(ions), ip(ifn))
        _check(rc, "qmc_jastrow_create")
        self._h = h

    def destroy(self):
        if self._h:
            _check(load_library().qmc_jastrow_destroy(self._h), "qmc_jastrow_destroy")
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def ratio(self, pos, iel, rnew, other=None, stream=None):
        """qmc_jastrow_ratio: (exp(-dJ), dJ) double [nw] for the move of electron iel of every walker to rnew [nw][3]."""
        nw, nel, _ = pos.shape
        ratio = torch.empty(nw, dtype=torch.float64, device=pos.device)
        dj = torch.empty(nw, dtype=torch.float64, device=pos.device)
        rc = load_library().qmc_jastrow_ratio(self._h, nw, nel, _dev(pos, torch.float64),
                                              0 if other is None else int(other.shape[1]), _dev(other, torch.float64, True),
                                              int(iel), _dev(rnew, torch.float64), _dev(ratio, None), _dev(dj, None), _stream(stream))
        _check(rc, "qmc_jastrow_ratio")
        return ratio, dj

    def value(self, pos, other=None, stream=None):
        """qmc_jastrow_value: J double [nw]."""
        nw, nel, _ = pos.shape
        out = torch.empty(nw, dtype=torch.float64, device=pos.device)
        rc = load_library().qmc_jastrow_value(self._h, nw, nel, _dev(pos, torch.float64),
                                              0 if other is None else int(other.shape[1]), _dev(other, torch.float64, True),
                                              _dev(out, None), _stream(stream))
        _check(rc, "qmc_jastrow_value")
        return out


class Wavefunction:
    """qmc_wf_t: Psi_T = D_up D_dn (eq. 26); does not own its determinants."""

    def __init__(self, det_up, det_dn):
        h = _vp()
        rc = load_library().qmc_wf_create(ctypes.byref(h), det_up._h, det_up.spline._h, det_dn._h, det_dn.spline._h)
        _check(rc, "qmc_wf_create")
        self._h, self.up, self.dn = h, det_up, det_dn
        self.nw, self.nup, self.ndn = det_up.nw, det_up.nel, det_dn.nel

    def destroy(self):
        if self._h:
            _check(load_library().qmc_wf_destroy(self._h), "qmc_wf_destroy")
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def sweep(self, pos_up, pos_dn, delta, unif, ratios_out=None, accept_out=None, forced_accept=None,
              fixed_node=False, force_out=None, drift_tau=0.0, jastrow=None, jratio_out=None, stream=None):
        """qmc_wf_sweep: delta [nsweeps][nup+ndn][nw][3], unif / outputs [nsweeps][nup+ndn][nw]."""
        n, nsweeps = self.nup + self.ndn, delta.shape[0]
        if tuple(delta.shape) != (nsweeps, n, self.nw, 3) or tuple(unif.shape) != (nsweeps, n, self.nw):
            raise QmcError("delta / unif shapes do not match the wavefunction")
        opts = None
        if fixed_node or force_out is not None or drift_tau or jastrow is not None:
            opts = ctypes.byref(SweepOpts(0, 0, None, 0, 1 if fixed_node else 0,
                                          None if force_out is None else _dev(force_out, torch.float64).value,
                                          float(drift_tau), None, None, None,
                                          None if jastrow is None else jastrow._h, None, 0,
                                          None if jratio_out is None else _dev(jratio_out, torch.float64).value))
        rc = load_library().qmc_wf_sweep(self._h, _dev(pos_up, torch.float64), _dev(pos_dn, torch.float64),
                                         _dev(delta, torch.float64), _dev(unif, torch.float64), nsweeps,
                                         _dev(ratios_out, torch.float64, True), _dev(accept_out, torch.uint8, True),
                                         _dev(forced_accept, torch.uint8, True), opts, _stream(stream))
        _check(rc, "qmc_wf_sweep")

    def kinetic(self, pos_up, pos_dn, stream=None):
        out = torch.empty(self.nw, dtype=torch.float64, device=pos_up.device)
        rc = load_library().qmc_wf_kinetic(self._h, _dev(pos_up, torch.float64), _dev(pos_dn, torch.float64),
                                           _dev(out, None), _stream(stream))
        _check(rc, "qmc_wf_kinetic")
        return out

    def get_stats(self, stream=None):
        """(log|Psi| double [nw], sign int32 [nw])."""
        dev = torch.device("cuda", torch.cuda.current_device())
        lp = torch.empty(self.nw, dtype=torch.float64, device=dev)
        sg = torch.empty(self.nw, dtype=torch.int32, device=dev)
        _check(load_library().qmc_wf_get_stats(self._h, _dev(lp, None), _dev(sg, None), _stream(stream)), "qmc_wf_get_stats")
        return lp, sg
