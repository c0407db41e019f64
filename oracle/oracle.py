"""ctypes front end of the CPU oracle (oracle/chem_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It marshals arguments; all arithmetic is in chem_oracle.c.  It imports
nothing from the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "chem_oracle.c")
_LIB = os.path.join(_HERE, "libchem_oracle.so")


def build(force: bool = False) -> str:
    """Compile chem_oracle.c with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


class _Mech(C.Structure):
    _fields_ = [("n_sp", C.c_int), ("n_rx", C.c_int),
                ("W", _dp), ("nasa_lo", _dp), ("nasa_hi", _dp), ("tmid", _dp),
                ("type", _ip),
                ("reac_ptr", _ip), ("reac_sp", _ip), ("reac_nu", _ip),
                ("prod_ptr", _ip), ("prod_sp", _ip), ("prod_nu", _ip),
                ("A", _dp), ("b", _dp), ("Ea", _dp),
                ("A0", _dp), ("b0", _dp), ("Ea0", _dp),
                ("troe", _dp),
                ("eff_ptr", _ip), ("eff_sp", _ip), ("eff_val", _dp)]


class RadauOpts(C.Structure):
    _fields_ = [("max_steps", C.c_int), ("newton_max", C.c_int), ("h0", C.c_double), ("fixed_steps", C.c_int),
                ("fd_jacobian", C.c_int)]


class RadauStats(C.Structure):
    _fields_ = [("status", C.c_int), ("nstep", C.c_int), ("naccpt", C.c_int), ("nrejct", C.c_int),
                ("nfcn", C.c_int), ("njac", C.c_int), ("ndec", C.c_int), ("nsol", C.c_int),
                ("nnewt_fail", C.c_int), ("h_last", C.c_double), ("err_last", C.c_double)]


STATS_DTYPE = np.dtype([("status", "i4"), ("nstep", "i4"), ("naccpt", "i4"), ("nrejct", "i4"),
                        ("nfcn", "i4"), ("njac", "i4"), ("ndec", "i4"), ("nsol", "i4"),
                        ("nnewt_fail", "i4"), ("_pad", "i4"), ("h_last", "f8"), ("err_last", "f8")])
assert STATS_DTYPE.itemsize == C.sizeof(RadauStats)

FCN = C.CFUNCTYPE(None, C.c_int, _dp, _dp, C.c_void_p)
JAC = C.CFUNCTYPE(None, C.c_int, _dp, _dp, C.c_void_p)

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_error_metric.restype = C.c_double
        _lib.orc_integrate.restype = C.c_int
        _lib.orc_lu_real.restype = C.c_int
        _lib.orc_lu_complex_ri.restype = C.c_int
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


class Mechanism:
    """Holds the numpy arrays of a synth mechanism dict alive and exposes the C struct."""

    def __init__(self, mech: dict):
        f64 = lambda k: np.ascontiguousarray(mech[k], dtype=np.float64)
        i32 = lambda k: np.ascontiguousarray(mech[k], dtype=np.int32)
        self.n_sp = int(mech["n_species"])
        self.n_rx = int(mech["n_reactions"])
        self._a = dict(W=f64("mol_weight"), nasa_lo=f64("nasa_lo"), nasa_hi=f64("nasa_hi"), tmid=f64("nasa_tmid"),
                       type=i32("rxn_type"), reac_ptr=i32("reac_ptr"), reac_sp=i32("reac_sp"), reac_nu=i32("reac_nu"),
                       prod_ptr=i32("prod_ptr"), prod_sp=i32("prod_sp"), prod_nu=i32("prod_nu"),
                       A=f64("arr_A"), b=f64("arr_b"), Ea=f64("arr_Ea"),
                       A0=f64("low_A"), b0=f64("low_b"), Ea0=f64("low_Ea"), troe=f64("troe"),
                       eff_ptr=i32("eff_ptr"), eff_sp=i32("eff_sp"), eff_val=f64("eff_val"))
        # ctypes needs a valid pointer even for empty arrays
        for k, v in self._a.items():
            if v.size == 0:
                self._a[k] = np.zeros(1, dtype=v.dtype)
        a = self._a
        self.c = _Mech(self.n_sp, self.n_rx, _d(a["W"]), _d(a["nasa_lo"]), _d(a["nasa_hi"]), _d(a["tmid"]),
                       _i(a["type"]), _i(a["reac_ptr"]), _i(a["reac_sp"]), _i(a["reac_nu"]),
                       _i(a["prod_ptr"]), _i(a["prod_sp"]), _i(a["prod_nu"]),
                       _d(a["A"]), _d(a["b"]), _d(a["Ea"]), _d(a["A0"]), _d(a["b0"]), _d(a["Ea0"]), _d(a["troe"]),
                       _i(a["eff_ptr"]), _i(a["eff_sp"]), _d(a["eff_val"]))

    # -- single-state routines -------------------------------------------------
    def thermo(self, T: float):
        cp, h, s = (np.empty(self.n_sp) for _ in range(3))
        lib().orc_thermo(C.byref(self.c), C.c_double(T), _d(cp), _d(h), _d(s))
        return cp, h, s

    def rates(self, P: float, y):
        y = np.ascontiguousarray(y, dtype=np.float64)
        Cc, wdot = np.empty(self.n_sp), np.empty(self.n_sp)
        kf, kr, q = (np.empty(self.n_rx) for _ in range(3))
        rho = C.c_double()
        lib().orc_rates(C.byref(self.c), C.c_double(P), _d(y), _d(Cc), _d(kf), _d(kr), _d(q), _d(wdot), C.byref(rho))
        return dict(C=Cc, kf=kf, kr=kr, q=q, wdot=wdot, rho=rho.value)

    def rhs(self, P: float, y):
        y = np.ascontiguousarray(y, dtype=np.float64)
        if y.ndim == 2:
            return np.stack([self.rhs(P, yy) for yy in y])
        f = np.empty(self.n_sp)
        lib().orc_rhs(C.byref(self.c), C.c_double(P), _d(y), _d(f))
        return f

    def jacobian(self, P: float, y):
        y = np.ascontiguousarray(y, dtype=np.float64)
        if y.ndim == 2:
            return np.stack([self.jacobian(P, yy) for yy in y])
        J = np.empty((self.n_sp, self.n_sp))
        lib().orc_jacobian(C.byref(self.c), C.c_double(P), _d(y), _d(J))
        return J

    # -- batched integration -----------------------------------------------------
    def integrate(self, y_in, P: float, t_end: float, rtol: float, atol: float, n_threads: int = 0,
                  h0: float = 0.0, max_steps: int = 0, fixed_steps: int = 0, fd_jacobian: int = 0):
        y_in = np.ascontiguousarray(y_in, dtype=np.float64)
        n = y_in.shape[0]
        assert y_in.shape[1] == self.n_sp
        y_out = np.empty_like(y_in)
        stats = np.zeros(n, dtype=STATS_DTYPE)
        opt = RadauOpts(max_steps, 0, h0, fixed_steps, fd_jacobian)
        used = lib().orc_integrate(C.byref(self.c), n, C.c_double(P), C.c_double(t_end), C.c_double(rtol),
                                   C.c_double(atol), _d(y_in), _d(y_out), C.byref(opt),
                                   stats.ctypes.data_as(C.c_void_p), n_threads)
        return y_out, stats, used


def radau5(f, jac, y0, t_end, rtol, atol, h0=0.0, max_steps=0, fixed_steps=0, newton_max=0, fd_jacobian=0):
    """Generic Radau IIA driver on a Python right-hand side f(y) and Jacobian jac(y) (row-major)."""
    y = np.array(y0, dtype=np.float64)
    n = y.size

    def _f(n_, yp, fp, _ctx):
        yy = np.ctypeslib.as_array(yp, shape=(n_,))
        np.ctypeslib.as_array(fp, shape=(n_,))[:] = f(yy)

    def _j(n_, yp, Jp, _ctx):
        yy = np.ctypeslib.as_array(yp, shape=(n_,))
        np.ctypeslib.as_array(Jp, shape=(n_ * n_,))[:] = np.asarray(jac(yy), dtype=np.float64).reshape(-1)

    opt = RadauOpts(max_steps, newton_max, h0, fixed_steps, fd_jacobian)
    st = RadauStats()
    lib().orc_radau5(n, FCN(_f), JAC(_j), None, _d(y), C.c_double(t_end), C.c_double(rtol), C.c_double(atol),
                     C.byref(opt), C.byref(st))
    return y, {k: getattr(st, k) for k, _ in RadauStats._fields_}


def radau_constants():
    out = np.empty(27)
    lib().orc_radau_constants(_d(out))
    return dict(T=out[0:9].reshape(3, 3).copy(), TI=out[9:18].reshape(3, 3).copy(), gamma=out[18], alpha=out[19],
                beta=out[20], c=out[21:24].copy(), dd=out[24:27].copy())


def lu_real(A):
    A = np.array(A, dtype=np.float64, order="C")
    ip = np.empty(A.shape[0], dtype=np.int32)
    ier = lib().orc_lu_real(A.shape[0], _d(A), _i(ip))
    return A, ip, ier


def lu_solve_real(LU, ip, b):
    b = np.array(b, dtype=np.float64)
    lib().orc_lu_solve_real(LU.shape[0], _d(LU), _i(ip), _d(b))
    return b


def lu_complex(A):
    A = np.array(A, dtype=np.complex128, order="C")
    ip = np.empty(A.shape[0], dtype=np.int32)
    ier = lib().orc_lu_complex_ri(A.shape[0], A.ctypes.data_as(_dp), _i(ip))
    return A, ip, ier


def lu_solve_complex(LU, ip, b):
    b = np.array(b, dtype=np.complex128)
    lib().orc_lu_solve_complex_ri(LU.shape[0], LU.ctypes.data_as(_dp), _i(ip), b.ctypes.data_as(_dp))
    return b


def error_metric(y, yhat, rtol, atol):
    """PAPER.md Eq. (1)-(2): returns (|E|, E_i)."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    yhat = np.ascontiguousarray(yhat, dtype=np.float64)
    E = np.empty(y.shape[0])
    Emax = lib().orc_error_metric(y.shape[0], y.shape[1], _d(y), _d(yhat), C.c_double(rtol), C.c_double(atol), _d(E))
    return Emax, E


def divergence(d):
    """PAPER.md Eq. (3) per group of 32 consecutive IVPs."""
    d = np.ascontiguousarray(d, dtype=np.int32)
    D = np.empty(d.size // 32)
    lib().orc_divergence(d.size, _i(d), _d(D))
    return D
