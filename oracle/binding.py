"""ctypes binding of oracle/libstreams_oracle.so (TEST INFRASTRUCTURE).

Argument marshalling only; every number comes out of streams_oracle.c.
"""
import ctypes as C

import numpy as np

from . import build as _build

_DBL = C.POINTER(C.c_double)


class OracleGrid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("pad_", C.c_int), ("len", C.c_double * 3)]


class OracleParams(C.Structure):
    _fields_ = [("gamma", C.c_double), ("Pr", C.c_double), ("Rgas", C.c_double), ("mu_ref", C.c_double),
                ("T_ref", C.c_double), ("visc_exp", C.c_double), ("suth_S", C.c_double),
                ("sensor_threshold", C.c_double), ("sensor_eps", C.c_double),
                ("T_wall", C.c_double * 2), ("y_wall", C.c_double * 2), ("fs", C.c_double * 5),
                ("shock_angle_deg", C.c_double), ("x_shock", C.c_double), ("cfl", C.c_double),
                ("dt_fixed", C.c_double),
                ("visc_model", C.c_int), ("order", C.c_int), ("weno_enable", C.c_int), ("forcing", C.c_int),
                ("viscous_enable", C.c_int), ("bc", C.c_int * 6), ("weno_order", C.c_int)]


class OracleDiag(C.Structure):
    _fields_ = [("step", C.c_longlong), ("time", C.c_double), ("dt", C.c_double), ("forcing", C.c_double),
                ("mass", C.c_double), ("mom", C.c_double * 3), ("energy", C.c_double), ("kinetic", C.c_double),
                ("volume", C.c_double), ("bulk_rhou", C.c_double),
                ("min_rho", C.c_double), ("min_p", C.c_double), ("max_mach", C.c_double), ("max_theta", C.c_double),
                ("max_speed", C.c_double * 3),
                ("weno_ifaces", C.c_longlong * 3), ("total_ifaces", C.c_longlong * 3),
                ("nonfinite", C.c_int), ("pad_", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.oracle_create.argtypes = [C.POINTER(OracleGrid), _DBL, _DBL, _DBL, C.POINTER(OracleParams),
                                    C.POINTER(C.c_void_p)]
        L.oracle_set_state.argtypes = [C.c_void_p, _DBL]
        L.oracle_get_state.argtypes = [C.c_void_p, _DBL]
        L.oracle_rhs.argtypes = [C.c_void_p, _DBL]
        L.oracle_rhs_parts.argtypes = [C.c_void_p, _DBL, _DBL]
        L.oracle_step.argtypes = [C.c_void_p, C.c_int]
        L.oracle_diagnostics.argtypes = [C.c_void_p, C.POINTER(OracleDiag)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_destroy.restype = None
        L.oracle_coeffs.argtypes = [C.c_int, _DBL, _DBL]
        L.oracle_weno5.argtypes = [C.c_double] * 5
        L.oracle_weno5.restype = C.c_double
        L.oracle_weno3.argtypes = [C.c_double] * 3
        L.oracle_weno3.restype = C.c_double
        L.oracle_eigen.argtypes = [C.c_int, C.c_double, _DBL, C.c_double, _DBL, _DBL, _DBL]
        L.oracle_eigen.restype = None
        L.oracle_shock_state.argtypes = [C.POINTER(OracleParams), _DBL, _DBL]
        L.oracle_get_metrics.argtypes = [C.c_void_p, C.c_int, _DBL, _DBL]
        L.oracle_get_sensor.argtypes = [C.c_void_p, _DBL, C.POINTER(C.c_ubyte)]
        L.oracle_get_prims.argtypes = [C.c_void_p, _DBL]
        L.oracle_stats_accumulate.argtypes = [C.c_void_p]
        L.oracle_stats_read.argtypes = [C.c_void_p, _DBL, C.POINTER(C.c_longlong)]
        L.oracle_stats_reset.argtypes = [C.c_void_p]
        L.oracle_get_ghosted.argtypes = [C.c_void_p, _DBL]
        L.oracle_roe_state.argtypes = [C.c_double, _DBL, C.c_double, C.c_double, _DBL, C.c_double, _DBL, _DBL]
        L.oracle_roe_state.restype = None
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_DBL)


def make_params(params: dict) -> OracleParams:
    """Fill the oracle's own parameter struct from the plain dict of a workload."""
    p = OracleParams()
    for name, _t in OracleParams._fields_:
        if name == "pad_":
            continue
        v = params.get("weno_order", 5) if name == "weno_order" else params[name]
        if isinstance(v, (list, tuple, np.ndarray)):
            arr = getattr(p, name)
            for i, x in enumerate(v):
                arr[i] = x
        else:
            setattr(p, name, v)
    return p


def coeffs(order):
    a = np.zeros(3)
    b = np.zeros(3)
    n = lib().oracle_coeffs(order, _p(a), _p(b))
    return n, a, b


def weno5(a, b, c, d, e):
    return lib().oracle_weno5(a, b, c, d, e)


def weno3(a, b, c):
    return lib().oracle_weno3(a, b, c)


def eigen(d, gamma, ubar, Hbar):
    ub = np.ascontiguousarray(ubar, dtype=np.float64)
    Lm = np.zeros((5, 5))
    Rm = np.zeros((5, 5))
    lam = np.zeros(5)
    lib().oracle_eigen(d, gamma, _p(ub), Hbar, _p(Lm), _p(Rm), _p(lam))
    return Lm, Rm, lam


def roe_state(rho_a, u_a, H_a, rho_b, u_b, H_b):
    ua = np.ascontiguousarray(u_a, dtype=np.float64)
    ub = np.ascontiguousarray(u_b, dtype=np.float64)
    out = np.zeros(3)
    Hb = C.c_double(0.0)
    lib().oracle_roe_state(rho_a, _p(ua), H_a, rho_b, _p(ub), H_b, _p(out), C.byref(Hb))
    return out, Hb.value


def shock_state(params: dict):
    p = make_params(params)
    post = np.zeros(5)
    beta = C.c_double(0.0)
    rc = lib().oracle_shock_state(C.byref(p), _p(post), C.byref(beta))
    if rc != 0:
        raise ValueError(f"oracle_shock_state failed: {rc}")
    return post, beta.value


class Oracle:
    """One oracle context: grid (nx,ny,nz,len), node coordinates, params dict."""

    def __init__(self, grid: dict, x, y, z, params: dict):
        self.n = (int(grid["nx"]), int(grid["ny"]), int(grid["nz"]))
        g = OracleGrid()
        g.nx, g.ny, g.nz = self.n
        for i in range(3):
            g.len[i] = grid["len"][i]
        self._x = [np.ascontiguousarray(a, dtype=np.float64) for a in (x, y, z)]
        self._params = make_params(params)
        h = C.c_void_p()
        rc = lib().oracle_create(C.byref(g), _p(self._x[0]), _p(self._x[1]), _p(self._x[2]),
                                 C.byref(self._params), C.byref(h))
        if rc != 0:
            raise ValueError(f"oracle_create failed: {rc}")
        self._h = h
        self.shape = (5, self.n[2], self.n[1], self.n[0])

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc, allow=()):
        if rc != 0 and rc not in allow:
            raise RuntimeError(f"oracle call failed: {rc}")
        return rc

    def set_state(self, w):
        w = np.ascontiguousarray(w, dtype=np.float64)
        assert w.shape == self.shape, (w.shape, self.shape)
        self._chk(lib().oracle_set_state(self._h, _p(w)))

    def get_state(self):
        w = np.empty(self.shape)
        self._chk(lib().oracle_get_state(self._h, _p(w)))
        return w

    def rhs(self):
        r = np.empty(self.shape)
        self._chk(lib().oracle_rhs(self._h, _p(r)))
        return r

    def rhs_parts(self):
        a = np.empty(self.shape)
        b = np.empty(self.shape)
        self._chk(lib().oracle_rhs_parts(self._h, _p(a), _p(b)))
        return a, b

    def step(self, n=1):
        self._chk(lib().oracle_step(self._h, int(n)))

    def diagnostics(self, check=True):
        d = OracleDiag()
        rc = lib().oracle_diagnostics(self._h, C.byref(d))
        self._chk(rc, allow=() if check else (-4,))
        return d

    def metrics(self, d):
        h = np.empty(self.n[d])
        g = np.empty(self.n[d])
        self._chk(lib().oracle_get_metrics(self._h, d, _p(h), _p(g)))
        return h, g

    def sensor(self):
        th = np.empty(self.shape[1:])
        fl = np.empty((3,) + self.shape[1:], dtype=np.uint8)
        self._chk(lib().oracle_get_sensor(self._h, _p(th), fl.ctypes.data_as(C.POINTER(C.c_ubyte))))
        return th, fl

    def stats_accumulate(self):
        self._chk(lib().oracle_stats_accumulate(self._h))

    def stats_read(self):
        """(profiles [16][ny], number of samples): rho,u,v,w,p,T,mu,rho u,rho v,rho w,rho T,rho uu,rho vv,rho ww,rho uv,TT"""
        out = np.empty((16, self.n[1]))
        n = C.c_longlong(0)
        self._chk(lib().oracle_stats_read(self._h, _p(out), C.byref(n)))
        return out, n.value

    def stats_reset(self):
        self._chk(lib().oracle_stats_reset(self._h))

    def ghosted(self):
        """Ghost-filled conservative state [5][nz+6][ny+6][nx+6] (S1)."""
        wg = np.empty((5, self.n[2] + 6, self.n[1] + 6, self.n[0] + 6))
        self._chk(lib().oracle_get_ghosted(self._h, _p(wg)))
        return wg

    def prims(self):
        q = np.empty((9,) + self.shape[1:])
        self._chk(lib().oracle_get_prims(self._h, _p(q)))
        return q


def threads():
    return lib().oracle_threads()
