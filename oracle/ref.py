"""ctypes binding of the ORACLE (oracle/libgrmhd_ref.so).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It shares nothing with the
CUDA path (paper_2406_11669_b200/).  All arrays are numpy, host memory, fp64.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "grmhd_ref.cpp")
_HDR = os.path.join(_HERE, "grmhd_ref.h")
_LIB = os.path.join(_HERE, "libgrmhd_ref.so")
G = 3


def build(force: bool = False) -> str:
    """Compile the oracle (plain g++, no FMA contraction)."""
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(_LIB) < os.path.getmtime(p) for p in (_SRC, _HDR))
    if force or stale:
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC",
               "-shared", "-o", _LIB, _SRC]
        subprocess.check_call(cmd)
    return _LIB


class RefOpts(C.Structure):
    _fields_ = [("gamma_ad", C.c_double), ("poly_k", C.c_double), ("poly_gamma", C.c_double),
                ("rho_atm", C.c_double), ("p_floor", C.c_double), ("w_max", C.c_double),
                ("c2p_tol", C.c_double), ("c2p_maxit", C.c_int), ("recon", C.c_int),
                ("ppm_flatten", C.c_int), ("riemann", C.c_int), ("rk", C.c_int),
                ("bc", C.c_int * 3)]


class RefStats(C.Structure):
    _fields_ = [("t", C.c_double), ("dt", C.c_double), ("maxspeed", C.c_double * 3),
                ("steps", C.c_longlong), ("c2p_fail", C.c_longlong), ("p_fix", C.c_longlong),
                ("atmo", C.c_longlong), ("w_cap", C.c_longlong), ("c2p_maxiter", C.c_longlong),
                ("c2p_backup", C.c_longlong)]


def make_opts(gamma_ad=5.0 / 3.0, poly_k=1.0, poly_gamma=None, rho_atm=1e-10, p_floor=1e-12,
              w_max=100.0, c2p_tol=1e-12, c2p_maxit=100, recon=1, ppm_flatten=1, riemann=0,
              rk=3, bc=(0, 0, 0)) -> RefOpts:
    o = RefOpts()
    o.gamma_ad = gamma_ad
    o.poly_k = poly_k
    o.poly_gamma = gamma_ad if poly_gamma is None else poly_gamma
    o.rho_atm = rho_atm
    o.p_floor = p_floor
    o.w_max = w_max
    o.c2p_tol = c2p_tol
    o.c2p_maxit = c2p_maxit
    o.recon = recon
    o.ppm_flatten = ppm_flatten
    o.riemann = riemann
    o.rk = rk
    for a in range(3):
        o.bc[a] = int(bc[a])
    return o


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.ref_get_num_threads.restype = C.c_int
    return _lib


def set_num_threads(n: int) -> None:
    lib().ref_set_num_threads(C.c_int(int(n)))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ptr_array(arrs, n):
    PA = C.POINTER(C.c_double) * n
    out = PA()
    for i, a in enumerate(arrs):
        if a is None:
            out[i] = None
        else:
            assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
            out[i] = _dp(a)
    return out


class RefSolver:
    """Handle-level oracle: same calls as the product's C ABI, host numpy arrays."""

    def __init__(self, nx, ny, nz, dx, opts: RefOpts):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.opts = opts
        self.h = C.c_void_p()
        d = (C.c_double * 3)(*[float(x) for x in dx])
        rc = lib().ref_create(self.nx, self.ny, self.nz, G, d, C.byref(opts), C.byref(self.h))
        if rc != 0:
            raise ValueError(f"ref_create failed: {rc}")
        self.cc_shape = (self.nz + 2 * G, self.ny + 2 * G, self.nx + 2 * G)
        self.st_shape = (self.nz + 2 * G + 1, self.ny + 2 * G + 1, self.nx + 2 * G + 1)

    def __del__(self):
        if getattr(self, "h", None) and self.h.value:
            lib().ref_destroy(self.h)
            self.h = C.c_void_p()

    @staticmethod
    def _chk(rc, what):
        if rc != 0:
            raise RuntimeError(f"{what} failed: {rc}")

    def set_metric(self, fields):
        fields = [np.ascontiguousarray(f, dtype=np.float64) for f in fields]
        assert len(fields) == 16 and all(f.shape == self.cc_shape for f in fields)
        self._chk(lib().ref_set_metric(self.h, _ptr_array(fields, 16)), "ref_set_metric")

    def set_prims(self, fields):
        fields = [None if f is None else np.ascontiguousarray(f, dtype=np.float64)
                  for f in fields]
        assert len(fields) == 8
        self._chk(lib().ref_set_prims(self.h, _ptr_array(fields, 8)), "ref_set_prims")

    def set_vecpot(self, fields):
        fields = [np.ascontiguousarray(f, dtype=np.float64) for f in fields]
        assert len(fields) == 3 and all(f.shape == self.st_shape for f in fields)
        self._chk(lib().ref_set_vecpot(self.h, _ptr_array(fields, 3)), "ref_set_vecpot")

    def set_mask(self, mask):
        if mask is None:
            self._chk(lib().ref_set_mask(self.h, None), "ref_set_mask")
            return
        m = np.ascontiguousarray(mask, dtype=np.uint8)
        assert m.shape == self.cc_shape
        self._chk(lib().ref_set_mask(self.h, m.ctypes.data_as(C.POINTER(C.c_ubyte))),
                  "ref_set_mask")

    def set_option(self, key, value):
        self._chk(lib().ref_set_option(self.h, key.encode(), C.c_double(value)), "ref_set_option")

    def step(self, n, cfl):
        self._chk(lib().ref_step(self.h, int(n), C.c_double(cfl)), "ref_step")

    def step_until(self, t_end, cfl):
        n = C.c_int(0)
        self._chk(lib().ref_step_until(self.h, C.c_double(t_end), C.c_double(cfl), C.byref(n)),
                  "ref_step_until")
        return n.value

    def _get(self, fn, n, shape):
        out = [np.zeros(shape) for _ in range(n)]
        self._chk(fn(self.h, _ptr_array(out, n)), fn.__name__)
        return out

    def get_prims(self):
        return self._get(lib().ref_get_prims, 8, self.cc_shape)

    def get_cons(self):
        return self._get(lib().ref_get_cons, 8, self.cc_shape)

    def get_vecpot(self):
        return self._get(lib().ref_get_vecpot, 3, self.st_shape)

    def get_psi(self):
        out = np.zeros(self.st_shape)
        self._chk(lib().ref_get_psi(self.h, _dp(out)), "ref_get_psi")
        return out

    def get_bface(self):
        return self._get(lib().ref_get_bface, 3, self.st_shape)

    def stats(self) -> dict:
        s = RefStats()
        rc = lib().ref_get_stats(self.h, C.byref(s))
        d = {k: getattr(s, k) for k, _ in RefStats._fields_ if k != "maxspeed"}
        d["maxspeed"] = [s.maxspeed[i] for i in range(3)]
        d["rc"] = rc
        return d

    def rhs(self):
        dU = [np.zeros(self.cc_shape) for _ in range(5)]
        dA = [np.zeros(self.st_shape) for _ in range(3)]
        self._chk(lib().ref_rhs(self.h, _ptr_array(dU, 5), _ptr_array(dA, 3)), "ref_rhs")
        return dU, dA

    def rhs_gauge(self):
        dA = [np.zeros(self.st_shape) for _ in range(3)]
        dPsi = np.zeros(self.st_shape)
        self._chk(lib().ref_rhs_gauge(self.h, _ptr_array(dA, 3), _dp(dPsi)), "ref_rhs_gauge")
        return dA, dPsi

    def fluxes(self):
        fl = [np.zeros(self.st_shape) for _ in range(24)]
        self._chk(lib().ref_fluxes(self.h, _ptr_array(fl, 24)), "ref_fluxes")
        return [[fl[d * 8 + r] for r in range(8)] for d in range(3)]


# ---- point functions --------------------------------------------------------------
def _v(x, n):
    a = np.ascontiguousarray(x, dtype=np.float64).reshape(-1)
    assert a.size == n
    return a


def prim2con_pt(prim, metric, gamma_ad):
    out = np.zeros(8)
    lib().ref_prim2con_pt(_dp(_v(prim, 8)), _dp(_v(metric, 10)), C.c_double(gamma_ad), _dp(out))
    return out


def con2prim_pt(cons, metric, opts: RefOpts, masked=0):
    p = np.zeros(5)
    u = np.zeros(5)
    it = C.c_int(0)
    bits = lib().ref_con2prim_pt(_dp(_v(cons, 8)), _dp(_v(metric, 10)), C.byref(opts),
                                 int(masked), _dp(p), _dp(u), C.byref(it))
    return p, u, bits, it.value


def con2prim_backup_pt(cons, metric, opts: RefOpts):
    """2-D scheme with the 1-D backup enabled; status bit 16 = recovered by the backup."""
    p = np.zeros(5)
    u = np.zeros(5)
    it = C.c_int(0)
    bits = lib().ref_con2prim_backup_pt(_dp(_v(cons, 8)), _dp(_v(metric, 10)), C.byref(opts),
                                        _dp(p), _dp(u), C.byref(it))
    return p, u, bits, it.value


def con2prim1d_pt(cons, metric, opts: RefOpts):
    """The 1-D scheme alone (eqs 42-45): (rho, v^i, p), status 0 / 2, Brent iterations."""
    p = np.zeros(5)
    it = C.c_int(0)
    st = lib().ref_con2prim1d_pt(_dp(_v(cons, 8)), _dp(_v(metric, 10)), C.byref(opts), _dp(p),
                                 C.byref(it))
    return p, st, it.value


def c2p1d_relations_pt(cons, metric, opts: RefOpts, x):
    """(W^ of eq. 44, eps^ of eq. 45, f of eq. 43) at a given x = h W."""
    out = np.zeros(3)
    lib().ref_c2p1d_relations_pt(_dp(_v(cons, 8)), _dp(_v(metric, 10)), C.byref(opts),
                                 C.c_double(x), _dp(out))
    return out


def flux_pt(d, prim, metric, gamma_ad):
    out = np.zeros(8)
    lib().ref_flux_pt(int(d), _dp(_v(prim, 8)), _dp(_v(metric, 10)), C.c_double(gamma_ad),
                      _dp(out))
    return out


def speeds_pt(d, prim, metric, gamma_ad):
    out = np.zeros(2)
    lib().ref_speeds_pt(int(d), _dp(_v(prim, 8)), _dp(_v(metric, 10)), C.c_double(gamma_ad),
                        _dp(out))
    return out


def riemann_pt(d, primL, primR, metric_face, opts: RefOpts):
    out = np.zeros(8)
    lib().ref_riemann_pt(int(d), _dp(_v(primL, 8)), _dp(_v(primR, 8)), _dp(_v(metric_face, 10)),
                         C.byref(opts), _dp(out))
    return out


def source_pt(prim, metric, K, dalpha, dbeta, dgam, gamma_ad):
    out = np.zeros(5)
    lib().ref_source_pt(_dp(_v(prim, 8)), _dp(_v(metric, 10)), _dp(_v(K, 6)), _dp(_v(dalpha, 3)),
                        _dp(_v(dbeta, 9)), _dp(_v(dgam, 18)), C.c_double(gamma_ad), _dp(out))
    return out


def recon_line(method, flatten, q, press=None, vnorm=None):
    q = _v(q, len(q))
    n = q.size
    qL = np.full(n + 1, np.nan)
    qR = np.full(n + 1, np.nan)
    pp = _dp(_v(press, n)) if press is not None else None
    vv = _dp(_v(vnorm, n)) if vnorm is not None else None
    lib().ref_recon_line(int(method), int(flatten), n, _dp(q), pp, vv, _dp(qL), _dp(qR))
    return qL, qR
