"""ctypes binding of oracle/libhzo.so (hzo.h).  Test infrastructure only; argument marshalling only."""
import ctypes as C
import os

import numpy as np

from . import build as _build

_dp = C.POINTER(C.c_double)


class OracleGrid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("bc", C.c_int * 3)]


class OracleParams(C.Structure):
    _fields_ = [("gamma_ad", C.c_double), ("rho_atm", C.c_double), ("p_atm", C.c_double),
                ("atm_tol", C.c_double), ("cleaning", C.c_int), ("kappa", C.c_double),
                ("c2p_maxit", C.c_int), ("c2p_tol", C.c_double), ("c2p_scheme", C.c_int), ("energy_var", C.c_int), ("recon", C.c_int)]

    @classmethod
    def default(cls, **kw):
        p = cls()
        lib().hzo_default_params(C.byref(p))
        for k, v in kw.items():
            if not hasattr(p, k):
                raise AttributeError(k)
            setattr(p, k, v)
        return p


class OracleDiag(C.Structure):
    _fields_ = [("sumD", C.c_double), ("sumSx", C.c_double), ("sumSy", C.c_double), ("sumSz", C.c_double),
                ("sumTau", C.c_double), ("sumBx", C.c_double), ("sumBy", C.c_double), ("sumBz", C.c_double),
                ("sumPsi", C.c_double), ("divB_max", C.c_double), ("divB_L1", C.c_double),
                ("max_speed_over_dx", C.c_double), ("c2p_fail", C.c_longlong), ("atm_reset", C.c_longlong),
                ("p_floor", C.c_longlong), ("c2p_maxit_seen", C.c_int)]

    def asdict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


_lib = None


def lib():
    global _lib
    if _lib is None:
        # HZO_LIB: another build of the same source, e.g. the sanitizer build (oracle/build.py --sanitize)
        path = os.environ.get("HZO_LIB") or _build.build()
        L = C.CDLL(os.path.abspath(path))
        L.hzo_prim2con_point.argtypes = [_dp, _dp, C.c_double, _dp]
        L.hzo_con2prim_point.argtypes = [_dp, _dp, C.POINTER(OracleParams), C.c_double, _dp, C.POINTER(C.c_int)]
        L.hzo_c2p_residual_point.argtypes = [C.c_double, _dp, _dp, C.c_double]
        L.hzo_c2p_residual_point.restype = C.c_double
        L.hzo_flux_point.argtypes = [C.c_int, _dp, _dp, C.c_double, C.c_int, _dp]
        L.hzo_wavespeed_point.argtypes = [C.c_int, _dp, _dp, C.c_double, C.c_int, _dp]
        L.hzo_mc_slope.argtypes = [C.c_double] * 3
        L.hzo_mc_slope.restype = C.c_double
        L.hzo_ppm_edges.argtypes = [_dp, _dp, _dp]
        L.hzo_ppm_edges.restype = None
        L.hzo_hlle_point.argtypes = [C.c_int, _dp, _dp, _dp, C.c_double, C.c_int, _dp]
        L.hzo_source_point.argtypes = [_dp, _dp, _dp, C.c_double, _dp]
        L.hzo_default_params.argtypes = [C.POINTER(OracleParams)]
        L.hzo_create.argtypes = [C.POINTER(OracleGrid), C.POINTER(OracleParams), C.POINTER(C.c_void_p)]
        L.hzo_destroy.argtypes = [C.c_void_p]
        L.hzo_set_metric.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.hzo_set_primitives.argtypes = [C.c_void_p, _dp]
        L.hzo_step.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.hzo_substeps.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.hzo_get_primitives.argtypes = [C.c_void_p, _dp]
        L.hzo_get_psi.argtypes = [C.c_void_p, _dp]
        L.hzo_get_conserved.argtypes = [C.c_void_p, _dp]
        L.hzo_get_rhs.argtypes = [C.c_void_p, _dp]
        L.hzo_diagnostics.argtypes = [C.c_void_p, C.POINTER(OracleDiag)]
        L.hzo_set_psi.argtypes = [C.c_void_p, _dp]
        L.hzo_padded_extent.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.hzo_get_padded.argtypes = [C.c_void_p, C.c_int, C.c_int, _dp]
        L.hzo_strerror.restype = C.c_char_p
        L.hzo_strerror.argtypes = [C.c_int]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _arr(x, n=None):
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    if n is not None and a.size != n:
        raise ValueError(f"expected {n} values, got {a.size}")
    return a


class OracleError(RuntimeError):
    pass


def _chk(rc):
    if rc != 0:
        raise OracleError(f"hzo error {rc}: {lib().hzo_strerror(rc).decode()}")


# ---- point functions ---------------------------------------------------------------------------
def prim2con_point(prim9, met10, gamma_ad):
    out = np.empty(9)
    lib().hzo_prim2con_point(_p(_arr(prim9, 9)), _p(_arr(met10, 10)), gamma_ad, _p(out))
    return out


def con2prim_point(cons9, met10, par, zguess=-1.0):
    out = np.full(9, np.nan)
    it = C.c_int(0)
    rc = lib().hzo_con2prim_point(_p(_arr(cons9, 9)), _p(_arr(met10, 10)), C.byref(par), zguess, _p(out), C.byref(it))
    return rc, out, it.value


def c2p_residual_point(Z, cons9, met10, gamma_ad):
    return lib().hzo_c2p_residual_point(Z, _p(_arr(cons9, 9)), _p(_arr(met10, 10)), gamma_ad)


def flux_point(d, prim9, met10, gamma_ad, cleaning):
    out = np.empty(9)
    lib().hzo_flux_point(d, _p(_arr(prim9, 9)), _p(_arr(met10, 10)), gamma_ad, cleaning, _p(out))
    return out


def wavespeed_point(d, prim9, met10, gamma_ad, cleaning):
    out = np.empty(2)
    lib().hzo_wavespeed_point(d, _p(_arr(prim9, 9)), _p(_arr(met10, 10)), gamma_ad, cleaning, _p(out))
    return out


def mc_slope(qm, q0, qp):
    return lib().hzo_mc_slope(qm, q0, qp)


def ppm_edges(q5):
    a, b = C.c_double(0), C.c_double(0)
    lib().hzo_ppm_edges(_p(_arr(q5, 5)), C.byref(a), C.byref(b))
    return a.value, b.value


def hlle_point(d, primL, primR, met10, gamma_ad, cleaning):
    out = np.empty(9)
    lib().hzo_hlle_point(d, _p(_arr(primL, 9)), _p(_arr(primR, 9)), _p(_arr(met10, 10)), gamma_ad, cleaning, _p(out))
    return out


def source_point(prim9, met10, dmet30, gamma_ad):
    out = np.empty(4)
    lib().hzo_source_point(_p(_arr(prim9, 9)), _p(_arr(met10, 10)), _p(_arr(dmet30, 30)), gamma_ad, _p(out))
    return out


def num_threads():
    return lib().hzo_num_threads()


# ---- grid API ----------------------------------------------------------------------------------
class Oracle:
    """One grid of the CPU oracle.  Arrays are numpy float64, shape (planes, nz, ny, nx)."""

    def __init__(self, n, h, bc, par=None):
        L = lib()
        g = OracleGrid(int(n[0]), int(n[1]), int(n[2]), float(h[0]), float(h[1]), float(h[2]),
                       (C.c_int * 3)(*[int(b) for b in bc]))
        self.n = tuple(int(x) for x in n)
        self.ncell = self.n[0] * self.n[1] * self.n[2]
        self.par = par if par is not None else OracleParams.default()
        h_ = C.c_void_p()
        _chk(L.hzo_create(C.byref(g), C.byref(self.par), C.byref(h_)))
        self._h = h_

    def close(self):
        if self._h:
            lib().hzo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _shape(self, planes):
        return (planes, self.n[2], self.n[1], self.n[0])

    def set_metric(self, alpha, beta3, gamma6):
        a, b, g = _arr(alpha, self.ncell), _arr(beta3, 3 * self.ncell), _arr(gamma6, 6 * self.ncell)
        _chk(lib().hzo_set_metric(self._h, _p(a), _p(b), _p(g)))

    def set_primitives(self, prim8):
        a = _arr(prim8, 8 * self.ncell)
        _chk(lib().hzo_set_primitives(self._h, _p(a)))

    def step(self, dt, n):
        _chk(lib().hzo_step(self._h, dt, n))

    def substeps(self, dt, nsub):
        _chk(lib().hzo_substeps(self._h, dt, nsub))

    def get_primitives(self):
        out = np.empty(self._shape(8))
        _chk(lib().hzo_get_primitives(self._h, _p(out)))
        return out

    def get_psi(self):
        out = np.empty(self._shape(1))
        _chk(lib().hzo_get_psi(self._h, _p(out)))
        return out[0]

    def get_conserved(self):
        out = np.empty(self._shape(9))
        _chk(lib().hzo_get_conserved(self._h, _p(out)))
        return out

    def get_rhs(self):
        out = np.empty(self._shape(9))
        _chk(lib().hzo_get_rhs(self._h, _p(out)))
        return out

    def set_psi(self, psi):
        """Test accessor: a manufactured cleaning scalar (the API's prim8 starts it at 0)."""
        a = _arr(psi, self.ncell)
        _chk(lib().hzo_set_psi(self._h, _p(a)))

    def get_padded(self, which, field):
        """Test accessor: one padded array with its ghost layers, shape (Nz, Ny, Nx), and the ghost widths
        (gx, gy, gz).  which = "prim" (9 fields) or "metric" (10 fields)."""
        N, g = (C.c_int * 3)(), (C.c_int * 3)()
        _chk(lib().hzo_padded_extent(self._h, N, g))
        out = np.empty((N[2], N[1], N[0]))
        _chk(lib().hzo_get_padded(self._h, {"prim": 0, "metric": 1}[which], int(field), _p(out)))
        return out, (g[0], g[1], g[2])

    def diagnostics(self):
        d = OracleDiag()
        _chk(lib().hzo_diagnostics(self._h, C.byref(d)))
        return d.asdict()
