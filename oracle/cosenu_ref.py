"""ctypes loader for oracle/libcosenu_ref.so (test infrastructure only; see cosenu_ref.h)."""
import ctypes as C
import os

import numpy as np

from . import build_oracle

FD4_KO3, FV_WENO7 = 0, 1
OPT_EPS_KO, OPT_WENO_EPS, OPT_ADVECT, OPT_THREADS, OPT_QUADRATURE, OPT_KO_ORDER = 0, 1, 2, 3, 4, 5


class Diag(C.Structure):
    _fields_ = [("t", C.c_double), ("step", C.c_int64),
                ("psurv_nu", C.c_double), ("psurv_nubar", C.c_double),
                ("dP_max", C.c_double), ("dP_avg", C.c_double),
                ("M0", C.c_double * 3), ("dM0", C.c_double * 3),
                ("trace_dev_max", C.c_double), ("ex_abs_max", C.c_double)]

    def asdict(self):
        return {"t": self.t, "step": self.step, "psurv_nu": self.psurv_nu,
                "psurv_nubar": self.psurv_nubar, "dP_max": self.dP_max, "dP_avg": self.dP_avg,
                "M0": list(self.M0), "dM0": list(self.dM0),
                "trace_dev_max": self.trace_dev_max, "ex_abs_max": self.ex_abs_max}


_lib = None


def lib():
    global _lib
    if _lib is None:
        # COSENU_REF_LIB: another build of the same source (the sanitizer build of tests/test_host_logic.py)
        path = os.environ.get("COSENU_REF_LIB") or build_oracle.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        L.cosenu_ref_create.restype = C.c_void_p
        L.cosenu_ref_create.argtypes = [C.c_int64, C.c_int32] + [C.c_double] * 5 + [C.c_int]
        L.cosenu_ref_set_option.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.cosenu_ref_init.argtypes = [C.c_void_p, C.c_uint64, C.c_double, C.c_double, C.c_double,
                                      C.c_double, C.c_int]
        L.cosenu_ref_set_state.argtypes = [C.c_void_p, dp, C.c_double]
        L.cosenu_ref_step.argtypes = [C.c_void_p, C.c_int64]
        L.cosenu_ref_get_state.argtypes = [C.c_void_p, dp]
        L.cosenu_ref_diagnostics.argtypes = [C.c_void_p, C.POINTER(Diag)]
        L.cosenu_ref_destroy.argtypes = [C.c_void_p]
        L.cosenu_ref_destroy.restype = None
        L.cosenu_ref_last_error.argtypes = [C.c_void_p]
        L.cosenu_ref_last_error.restype = C.c_char_p
        L.cosenu_ref_rhs.argtypes = [C.c_void_p, dp, dp]
        L.cosenu_ref_moments.argtypes = [C.c_void_p, dp, dp]
        L.cosenu_ref_weno7_candidates.argtypes = [dp, dp]
        L.cosenu_ref_weno7_candidates.restype = None
        L.cosenu_ref_weno7_si.argtypes = [dp, dp]
        L.cosenu_ref_weno7_si.restype = None
        L.cosenu_ref_weno7_dr.argtypes = [dp]
        L.cosenu_ref_weno7_dr.restype = None
        L.cosenu_ref_weno7_face.argtypes = [dp, C.c_double]
        L.cosenu_ref_weno7_face.restype = C.c_double
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class RefSim:
    """Thin wrapper over the cosenu_ref_* C ABI (same call names as the product binding)."""

    def __init__(self, nz, nv, L, dt, omega, theta, mu, scheme, eps_ko=None, weno_eps=None,
                 advect=True, threads=0, quadrature=0, ko_order=2):
        self._L = lib()
        self.nz, self.nv = int(nz), int(nv)
        self.h = self._L.cosenu_ref_create(nz, nv, L, dt, omega, theta, mu, scheme)
        if not self.h:
            raise ValueError(self._L.cosenu_ref_last_error(None).decode())
        if eps_ko is not None:
            self.set_option(OPT_EPS_KO, eps_ko)
        if weno_eps is not None:
            self.set_option(OPT_WENO_EPS, weno_eps)
        if not advect:
            self.set_option(OPT_ADVECT, 0)
        if threads:
            self.set_option(OPT_THREADS, threads)
        if quadrature:
            self.set_option(OPT_QUADRATURE, quadrature)
        if ko_order != 2:
            self.set_option(OPT_KO_ORDER, ko_order)

    def _chk(self, rc):
        if rc != 0:
            raise RuntimeError("cosenu_ref error %d: %s" % (rc, self._L.cosenu_ref_last_error(self.h).decode()))

    def set_option(self, key, value):
        self._chk(self._L.cosenu_ref_set_option(self.h, key, float(value)))

    def init(self, seed, sigma_nu=0.6, sigma_nubar=0.5, alpha=0.9, pert_amp=1e-6, pert_kind=0):
        self._chk(self._L.cosenu_ref_init(self.h, seed, sigma_nu, sigma_nubar, alpha, pert_amp, pert_kind))

    def set_state(self, state, t=0.0):
        a = np.ascontiguousarray(state, dtype=np.float64)
        assert a.shape == (8, self.nz, self.nv)
        self._chk(self._L.cosenu_ref_set_state(self.h, _p(a), t))

    def step(self, n=1):
        self._chk(self._L.cosenu_ref_step(self.h, n))

    def get_state(self):
        out = np.empty((8, self.nz, self.nv), dtype=np.float64)
        self._chk(self._L.cosenu_ref_get_state(self.h, _p(out)))
        return out

    def diagnostics(self):
        d = Diag()
        self._chk(self._L.cosenu_ref_diagnostics(self.h, C.byref(d)))
        return d.asdict()

    def rhs(self, y):
        a = np.ascontiguousarray(y, dtype=np.float64)
        assert a.shape == (8, self.nz, self.nv)
        k = np.empty_like(a)
        self._chk(self._L.cosenu_ref_rhs(self.h, _p(a), _p(k)))
        return k

    def moments(self, y):
        a = np.ascontiguousarray(y, dtype=np.float64)
        out = np.empty((6, self.nz), dtype=np.float64)
        self._chk(self._L.cosenu_ref_moments(self.h, _p(a), _p(out)))
        return out

    def close(self):
        if self.h:
            self._L.cosenu_ref_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def weno7_candidates(f):
    f = np.ascontiguousarray(f, dtype=np.float64); out = np.empty(4)
    lib().cosenu_ref_weno7_candidates(_p(f), _p(out)); return out


def weno7_si(f):
    f = np.ascontiguousarray(f, dtype=np.float64); out = np.empty(4)
    lib().cosenu_ref_weno7_si(_p(f), _p(out)); return out


def weno7_dr():
    out = np.empty(4); lib().cosenu_ref_weno7_dr(_p(out)); return out


def weno7_face(f, eps):
    f = np.ascontiguousarray(f, dtype=np.float64)
    return lib().cosenu_ref_weno7_face(_p(f), float(eps))
