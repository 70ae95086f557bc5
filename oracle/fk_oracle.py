"""ctypes binding of the CPU oracle (oracle/fk_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It never imports the CUDA package's
binding or kernels; the only thing it accepts from paper_2104_14561_b200 is a `Workload`
object (inputs) handed in by the caller.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fk_oracle.cpp")
_LIB = os.path.join(_HERE, "libfk_oracle.so")


def build(force: bool = False) -> str:
    """g++ -O2 -fopenmp -ffp-contract=off -> oracle/libfk_oracle.so (rebuilt when stale)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


class _Problem(C.Structure):
    _fields_ = [("d", C.c_int), ("n", C.c_int * 3), ("x", C.POINTER(C.c_double) * 3),
                ("dt", C.c_double), ("Q", C.c_int * 3), ("face_kind", (C.c_int * 2) * 3),
                ("face_value", (C.c_double * 2) * 3), ("slope_rule", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        pp = C.POINTER(_Problem)
        _lib.ofk_gauss_hermite.argtypes = [C.c_int, dp, dp]
        _lib.ofk_chi.argtypes = [pp, dp]
        _lib.ofk_pchip_slopes.argtypes = [C.c_int, dp, dp, C.c_long, dp]
        _lib.ofk_pchip_slopes_ex.argtypes = [C.c_int, dp, dp, C.c_long, dp, C.c_int, C.c_int]
        _lib.ofk_reduce.argtypes = [C.c_long, C.c_int, dp, dp, dp]
        _lib.ofk_interp.argtypes = [pp, dp, C.c_long, dp, dp]
        _lib.ofk_apply.argtypes = [pp, dp, dp, dp, dp]
        _lib.ofk_column.argtypes = [pp, dp, dp, C.c_int, C.c_int, dp]
        _lib.ofk_algorithm1.argtypes = [pp, dp, dp, C.c_int, C.c_int, dp]
        _lib.ofk_num_threads.restype = C.c_int
        _lib.ofk_set_num_threads.argtypes = [C.c_int]
        # virtual cores of these boxes are hyper-threads: half of them is the faster setting;
        # FK_ORACLE_THREADS overrides.  Reported as `cores` by bench.py.
        t = int(os.environ.get("FK_ORACLE_THREADS", "0")) or max(1, (os.cpu_count() or 2) // 2)
        _lib.ofk_set_num_threads(t)
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    """The scheme on one workload (grid, dt, Q, faces); coefficients are passed per call."""

    def __init__(self, wl):
        self.wl = wl
        self._x = [_f64(a) for a in wl.x]
        p = _Problem()
        p.d = wl.d
        for k in range(wl.d):
            p.n[k] = len(self._x[k])
            p.x[k] = _ptr(self._x[k])
            p.Q[k] = int(wl.Q[k])
            for s in range(2):
                p.face_kind[k][s] = int(wl.face_kind[k][s])
                p.face_value[k][s] = float(wl.face_value[k][s])
        p.dt = float(wl.dt)
        p.slope_rule = int(getattr(wl, "slope_rule", 0))
        self.p = p
        self.J = wl.J

    def chi(self):
        out = np.empty(self.J)
        lib().ofk_chi(C.byref(self.p), _ptr(out))
        return out

    def interp(self, u, pts):
        u = _f64(u)
        pts = _f64(pts).reshape(-1, self.wl.d)
        out = np.empty(len(pts))
        lib().ofk_interp(C.byref(self.p), _ptr(u), len(pts), _ptr(pts), _ptr(out))
        return out

    def apply(self, b, sigma, u):
        """One operator application (Scheme 1 steps 1-3) to the field u[J]."""
        b, sigma, u = _f64(b).reshape(-1), _f64(sigma).reshape(-1), _f64(u)
        assert b.size == self.wl.d * self.J and sigma.size == b.size and u.size == self.J
        out = np.empty(self.J)
        lib().ofk_apply(C.byref(self.p), _ptr(b), _ptr(sigma), _ptr(u), _ptr(out))
        return out

    def column(self, m):
        """Eq. 29: P(t_m, .) by m applications to chi; coefficients from the workload."""
        if self.wl.autonomous:
            b, s = self.wl.coeffs(0)
            b, s = _f64(b), _f64(s)
            auto = 1
        else:
            b, s = self.wl.coeff_table(0, max(m, 1))
            auto = 0
        out = np.empty(self.J)
        lib().ofk_column(C.byref(self.p), _ptr(b), _ptr(s), auto, int(m), _ptr(out))
        return out

    def column_streamed(self, m):
        """Same as column(m) without materialising the coefficient table (long columns)."""
        u = self.chi()
        for nu in range(m - 1, -1, -1):
            b, s = self.wl.coeffs(nu)
            u = self.apply(b, s, u)
        return u

    def algorithm1(self, N=None):
        """Algorithm 1 for the first N steps: returns P[N+1][J], row m = P(t_m, .)."""
        N = self.wl.N if N is None else int(N)
        if self.wl.autonomous:
            b, s = self.wl.coeffs(0)
            b, s = _f64(b), _f64(s)
            auto = 1
        else:
            b, s = self.wl.coeff_table(0, max(N, 1))
            auto = 0
        P = np.empty((N + 1, self.J))
        lib().ofk_algorithm1(C.byref(self.p), _ptr(b), _ptr(s), auto, N, _ptr(P))
        return P


def gauss_hermite(Q):
    a = np.empty(Q)
    w = np.empty(Q)
    rc = lib().ofk_gauss_hermite(int(Q), _ptr(a), _ptr(w))
    if rc:
        raise ValueError("Q out of range")
    return a, w


def reduce(P, w):
    """sum_j w_j P[m][j] for every row m of P."""
    P, w = _f64(P), _f64(w)
    P = P.reshape(-1, w.size)
    out = np.empty(P.shape[0])
    lib().ofk_reduce(w.size, P.shape[0], _ptr(P), _ptr(w), _ptr(out))
    return out


def pchip_slopes(x, u, periodic=False, weighted=False):
    x, u = _f64(x), _f64(u)
    du = np.empty_like(u)
    rc = lib().ofk_pchip_slopes_ex(len(x), _ptr(x), _ptr(u), 1, _ptr(du), int(periodic), int(weighted))
    if rc:
        raise ValueError("need at least 3 nodes")
    return du


def num_threads():
    return int(lib().ofk_num_threads())


def set_num_threads(t):
    lib().ofk_set_num_threads(int(t))
