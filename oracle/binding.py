"""ctypes binding of the CPU oracle (oracle/libprs_ref.so).  TEST INFRASTRUCTURE ONLY.

Mirrors prs_ref.h one to one; numpy arrays carry the fields (dense T[N^dims], x fastest).
"""
import ctypes as C

import numpy as np

from . import build as _build

F32, F64 = 0, 1
ARITH_LITERAL, ARITH_COEF, ARITH_FMA = 0, 1, 2
_DT = {F32: np.float32, F64: np.float64}


class Diag(C.Structure):
    _fields_ = [("step", C.c_int64), ("eta", C.c_double), ("link_count", C.c_uint64),
                ("wall_sites", C.c_uint64), ("sum_ratio", C.c_double), ("rho", C.c_double),
                ("gv2", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp, i64, dbl, u64, ci = C.c_void_p, C.c_int64, C.c_double, C.c_uint64, C.c_int
        L.prs_ref_create.argtypes = [C.POINTER(vp), ci, i64, ci, dbl, dbl, dbl, dbl, dbl, u64]
        L.prs_ref_destroy.argtypes = [vp]
        L.prs_ref_set_arith.argtypes = [vp, ci]
        L.prs_ref_set_beta.argtypes = [vp, dbl]
        L.prs_ref_scalars_beta.argtypes = [dbl, dbl, dbl, dbl, dbl, dbl, dbl, i64, C.POINTER(dbl)]
        L.prs_ref_set_threads.argtypes = [vp, ci]
        L.prs_ref_init.argtypes = [vp, dbl]
        L.prs_ref_step.argtypes = [vp, i64]
        L.prs_ref_diagnostics.argtypes = [vp, C.POINTER(Diag)]
        L.prs_ref_copy_out.argtypes = [vp, vp, vp]
        L.prs_ref_copy_in.argtypes = [vp, vp, vp, dbl, i64]
        L.prs_ref_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32),
                                            C.POINTER(C.c_uint32)]
        L.prs_ref_philox4x32_10.restype = None
        L.prs_ref_init_value.argtypes = [u64, u64, dbl]
        L.prs_ref_init_value.restype = dbl
        L.prs_ref_diagnostics_of.argtypes = [ci, i64, ci, vp, vp, dbl, dbl, C.POINTER(Diag)]
        L.prs_ref_step_sites.argtypes = [ci, i64, ci, ci, dbl, dbl, dbl, dbl, dbl, dbl, i64,
                                         vp, vp, vp, i64, vp, vp]
        L.prs_ref_scalars.argtypes = [dbl, dbl, dbl, dbl, dbl, dbl, i64, C.POINTER(dbl)]
        L.prs_ref_weighted_area_of.argtypes = [ci, i64, ci, vp, C.POINTER(dbl)]
        _lib = L
    return _lib


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError("%s failed with status %d" % (what, rc))


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


class RefSim:
    """One oracle simulation; same call names as the product binding."""

    def __init__(self, dims, N, precision=F32, alpha=3.0, era_m=1.0, deta=0.1, W0=10.0, phi0=1.0,
                 seed=1, arith=ARITH_LITERAL, threads=1, beta=0.0):
        self.dims, self.N, self.precision = dims, int(N), precision
        self.params = dict(alpha=alpha, era_m=era_m, deta=deta, W0=W0, phi0=phi0)
        self.dtype = _DT[precision]
        self.shape = (self.N,) * dims
        self._h = C.c_void_p()
        _chk(lib().prs_ref_create(C.byref(self._h), dims, self.N, precision, alpha, era_m, deta, W0,
                                  phi0, seed), "prs_ref_create")
        _chk(lib().prs_ref_set_arith(self._h, arith), "prs_ref_set_arith")
        _chk(lib().prs_ref_set_threads(self._h, threads), "prs_ref_set_threads")
        _chk(lib().prs_ref_set_beta(self._h, beta), "prs_ref_set_beta")

    def close(self):
        if self._h:
            lib().prs_ref_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def init(self, eta0=1.0):
        _chk(lib().prs_ref_init(self._h, eta0), "prs_ref_init")

    def step(self, nsteps=1):
        _chk(lib().prs_ref_step(self._h, nsteps), "prs_ref_step")

    def diagnostics(self):
        d = Diag()
        _chk(lib().prs_ref_diagnostics(self._h, C.byref(d)), "prs_ref_diagnostics")
        return d.as_dict()

    def copy_out(self):
        phi = np.empty(self.shape, self.dtype)
        pd = np.empty(self.shape, self.dtype)
        _chk(lib().prs_ref_copy_out(self._h, _ptr(phi), _ptr(pd)), "prs_ref_copy_out")
        return phi, pd

    def copy_in(self, phi, phidot, eta0=1.0, step=0):
        phi = np.ascontiguousarray(phi, self.dtype)
        phidot = np.ascontiguousarray(phidot, self.dtype)
        assert phi.shape == self.shape and phidot.shape == self.shape
        _chk(lib().prs_ref_copy_in(self._h, _ptr(phi), _ptr(phidot), eta0, step), "prs_ref_copy_in")


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().prs_ref_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


def init_value(seed, s, phi0=1.0):
    return float(lib().prs_ref_init_value(seed, s, phi0))


def diagnostics_of(phi, phidot, W0=10.0, phi0=1.0):
    phi = np.ascontiguousarray(phi)
    phidot = np.ascontiguousarray(phidot, phi.dtype)
    prec = F32 if phi.dtype == np.float32 else F64
    assert phi.dtype in (np.float32, np.float64) and phi.shape == phidot.shape
    d = Diag()
    _chk(lib().prs_ref_diagnostics_of(phi.ndim, phi.shape[0], prec, _ptr(phi), _ptr(phidot), W0, phi0,
                                      C.byref(d)), "prs_ref_diagnostics_of")
    return d.as_dict()


def weighted_area_of(phi):
    """Eq. 7 as printed: sum over crossing links of |grad phi| / sum |grad phi components| (double)."""
    phi = np.ascontiguousarray(phi)
    assert phi.dtype in (np.float32, np.float64)
    prec = F32 if phi.dtype == np.float32 else F64
    out = C.c_double()
    _chk(lib().prs_ref_weighted_area_of(phi.ndim, phi.shape[0], prec, _ptr(phi), C.byref(out)), "prs_ref_weighted_area_of")
    return float(out.value)


def step_sites(phi, phidot, sites, n, eta0=1.0, arith=ARITH_LITERAL, alpha=3.0, era_m=1.0, deta=0.1,
               W0=10.0, phi0=1.0):
    """phi^{n+1}, phidot^{n+1/2} at the listed linear site indices of a caller-held state."""
    assert phi.flags.c_contiguous and phidot.flags.c_contiguous and phi.dtype == phidot.dtype
    prec = F32 if phi.dtype == np.float32 else F64
    sites = np.ascontiguousarray(sites, np.int64)
    po = np.empty(sites.shape, phi.dtype)
    vo = np.empty(sites.shape, phi.dtype)
    _chk(lib().prs_ref_step_sites(phi.ndim, phi.shape[0], prec, arith, alpha, era_m, deta, W0, phi0,
                                  eta0, n, _ptr(phi), _ptr(phidot), _ptr(sites), sites.size,
                                  _ptr(po), _ptr(vo)), "prs_ref_step_sites")
    return po, vo


def scalars(n, eta0=1.0, alpha=3.0, era_m=1.0, deta=0.1, W0=10.0, phi0=1.0, beta=0.0):
    out = (C.c_double * 7)()
    _chk(lib().prs_ref_scalars_beta(alpha, beta, era_m, deta, W0, phi0, eta0, n, out), "prs_ref_scalars_beta")
    return dict(zip(("eta", "delta", "A", "B", "V0", "K", "I"), [float(v) for v in out]))
