"""Thin Python binding of include/chem.h (libchem.so).  Argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; PyTorch is used for device memory and
streams.  There is no CPU fallback: if libchem.so is missing or no CUDA device is present, the
calls raise.  This module never imports anything under oracle/.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libchem.so")

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class ChemError(RuntimeError):
    pass


class chem_mech_desc(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_reactions", C.c_int32),
                ("mol_weight", _dp), ("nasa_lo", _dp), ("nasa_hi", _dp), ("nasa_tmid", _dp),
                ("rxn_type", _ip), ("reac_ptr", _ip), ("reac_sp", _ip), ("reac_nu", _ip),
                ("prod_ptr", _ip), ("prod_sp", _ip), ("prod_nu", _ip),
                ("arr_A", _dp), ("arr_b", _dp), ("arr_Ea", _dp),
                ("low_A", _dp), ("low_b", _dp), ("low_Ea", _dp), ("troe", _dp),
                ("eff_ptr", _ip), ("eff_sp", _ip), ("eff_val", _dp)]


class chem_opts(C.Structure):
    _fields_ = [("h0", C.c_double), ("max_steps", C.c_int32), ("newton_max", C.c_int32),
                ("kernel", C.c_int32), ("reorder", C.c_int32), ("P_per_state", C.c_void_p), ("cost_hint", C.c_void_p),
                ("fd_jacobian", C.c_int32), ("fixed_steps", C.c_int32)]


STATS_DTYPE = np.dtype([("status", "i4"), ("nstep", "i4"), ("naccpt", "i4"), ("nrejct", "i4"), ("nfcn", "i4"),
                        ("njac", "i4"), ("ndec", "i4"), ("nsol", "i4"), ("nnewt_fail", "i4"), ("reserved", "i4"),
                        ("h_last", "f8")])
assert STATS_DTYPE.itemsize == 48

EXPORTS = ["chem_mech_load", "chem_mech_free", "chem_mech_info", "chem_rhs", "chem_jacobian", "chem_lu_solve",
           "chem_integrate", "chem_integrate_ex", "chem_integrate_host", "chem_launch_count", "chem_flop_model",
           "chem_last_error", "chem_last_kernel", "chem_fp64_probe", "chem_tps_radau_solve", "chem_integrate_noalloc", "chem_scratch_trim", "chem_flop_model_t1"]

_lib = None


def lib():
    """Load libchem.so (built in-tree by paper_1607_03884_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ChemError(f"{LIB_PATH} is missing: run `python -m paper_1607_03884_b200.build` "
                            "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.chem_last_error.restype = C.c_char_p
        L.chem_launch_count.restype = C.c_int64
        L.chem_mech_load.argtypes = [C.POINTER(chem_mech_desc), C.POINTER(C.c_void_p)]
        L.chem_mech_free.argtypes = [C.c_void_p]
        L.chem_mech_free.restype = None
        L.chem_mech_info.argtypes = [C.c_void_p, _ip, _ip]
        L.chem_rhs.argtypes = [C.c_void_p, C.c_int32, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.chem_jacobian.argtypes = [C.c_void_p, C.c_int32, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.chem_lu_solve.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_void_p]
        L.chem_integrate.argtypes = [C.c_void_p, C.c_int32, C.c_double, C.c_double, C.c_double, C.c_double,
                                     C.c_void_p, C.c_void_p, C.c_void_p]
        L.chem_integrate_ex.argtypes = [C.c_void_p, C.c_int32, C.c_double, C.c_double, C.c_double, C.c_double,
                                        C.c_void_p, C.c_void_p, C.POINTER(chem_opts), C.c_void_p, C.c_void_p]
        L.chem_integrate_noalloc.argtypes = L.chem_integrate_ex.argtypes
        L.chem_integrate_host.argtypes = [C.c_void_p, C.c_int32, C.c_double, C.c_double, C.c_double, C.c_double,
                                          C.c_void_p, C.c_void_p, C.POINTER(chem_opts), C.c_void_p]
        L.chem_flop_model.argtypes = [C.c_void_p, _dp]
        L.chem_flop_model_t1.argtypes = [C.c_void_p, _dp]
        L.chem_last_kernel.argtypes = [C.c_void_p]
        L.chem_fp64_probe.argtypes = [C.c_int32, C.c_int32, _dp]
        L.chem_tps_radau_solve.argtypes = [C.c_int32, C.c_int32, C.c_void_p, C.c_double, C.c_double, C.c_double,
                                           C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise ChemError(f"libchem error {rc}: {lib().chem_last_error().decode()}")


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _dev_f64(t, shape=None):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise ChemError("expected a contiguous float64 CUDA tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ChemError(f"expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return C.c_void_p(t.data_ptr())


class Mechanism:
    """Owner of a `chem_mech*` (device tables).  `desc` is a synth-style dict of numpy arrays."""

    def __init__(self, desc: dict):
        f64 = lambda k: np.ascontiguousarray(desc[k], dtype=np.float64)
        i32 = lambda k: np.ascontiguousarray(desc[k], dtype=np.int32)
        keep = {}
        d = chem_mech_desc()
        d.n_species = int(desc["n_species"])
        d.n_reactions = int(desc["n_reactions"])
        for name, ctype in chem_mech_desc._fields_[2:]:
            a = f64(name) if ctype is _dp else i32(name)
            if a.size == 0:
                a = np.zeros(1, dtype=a.dtype)
            keep[name] = a
            setattr(d, name, a.ctypes.data_as(ctype))
        self._h = C.c_void_p()
        _check(lib().chem_mech_load(C.byref(d), C.byref(self._h)))
        self.n_species = d.n_species
        self.n_reactions = d.n_reactions

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().chem_mech_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def flop_model(self, transcendental_1=False):
        """algorithmic flops per operation; exp/log/pow/sqrt count 20 each (the roofline convention) or 1 each"""
        out = np.empty(5)
        _check((lib().chem_flop_model_t1 if transcendental_1 else lib().chem_flop_model)(self._h, out.ctypes.data_as(_dp)))
        return dict(rhs=out[0], jac=out[1], lu=out[2], newton=out[3], err=out[4])


def chem_mech_load(desc: dict) -> Mechanism:
    return Mechanism(desc)


def chem_rhs(mech: Mechanism, P: float, y, stream=None):
    import torch
    n = y.shape[0]
    f = torch.empty_like(y)
    _check(lib().chem_rhs(mech._h, n, P, _dev_f64(y, (n, mech.n_species)), _dev_f64(f), _stream_ptr(stream)))
    return f


def chem_jacobian(mech: Mechanism, P: float, y, stream=None):
    import torch
    n, N = y.shape[0], mech.n_species
    J = torch.empty((n, N, N), dtype=torch.float64, device=y.device)
    _check(lib().chem_jacobian(mech._h, n, P, _dev_f64(y, (n, N)), _dev_f64(J), _stream_ptr(stream)))
    return J


def chem_lu_solve(A, b, stream=None):
    """A: [batch, n, n] float64 or complex128 CUDA tensor, b: [batch, n].  Returns (x, info)."""
    import torch
    cplx = A.is_complex()
    batch, n = A.shape[0], A.shape[1]
    Ar = torch.view_as_real(A.contiguous()).contiguous() if cplx else A.contiguous()
    br = torch.view_as_real(b.contiguous()).contiguous() if cplx else b.contiguous()
    x = torch.empty_like(br)
    info = torch.empty(max(batch, 1), dtype=torch.int32, device=A.device)
    _check(lib().chem_lu_solve(n, batch, int(cplx), C.c_void_p(Ar.data_ptr()), C.c_void_p(br.data_ptr()),
                               C.c_void_p(x.data_ptr()), C.c_void_p(info.data_ptr()), _stream_ptr(stream)))
    return (torch.view_as_complex(x) if cplx else x), info[:batch]


def chem_tps_radau_solve(J, fac1: float, alphn: float, betan: float, b, stream=None):
    """Thread-per-state linear algebra hook (include/chem.h).  J: [batch, n, n], b: [batch, 3, n] float64 CUDA tensors.
    Returns (x [batch, 3, n], info [batch])."""
    import torch
    batch, n = J.shape[0], J.shape[1]
    x = torch.zeros_like(b)
    info = torch.empty(max(batch, 1), dtype=torch.int32, device=J.device)
    _check(lib().chem_tps_radau_solve(n, batch, _dev_f64(J, (batch, n, n)), fac1, alphn, betan, _dev_f64(b, (batch, 3, n)),
                                      _dev_f64(x), C.c_void_p(info.data_ptr()), _stream_ptr(stream)))
    return x, info[:batch]


def _opts(h0=0.0, max_steps=0, newton_max=0, kernel=0, reorder=0, P_per_state=None, cost_hint=None, fd_jacobian=0, fixed_steps=0):
    """cost_hint: int32 CUDA tensor [n_states] (e.g. nstep of the previous global step); used when reorder=1"""
    o = chem_opts()
    o.h0, o.max_steps, o.newton_max, o.kernel, o.reorder = h0, max_steps, newton_max, kernel, reorder
    o.P_per_state = P_per_state.data_ptr() if P_per_state is not None else None
    o.cost_hint = cost_hint.data_ptr() if cost_hint is not None else None
    o.fd_jacobian = fd_jacobian
    o.fixed_steps = fixed_steps
    return o


def chem_integrate(mech: Mechanism, P: float, t_end: float, rtol: float, atol: float, y_in, y_out=None, stream=None):
    """The hot path (device tensors).  Returns y_out."""
    import torch
    n = y_in.shape[0]
    if y_out is None:
        y_out = torch.empty_like(y_in)
    _check(lib().chem_integrate(mech._h, n, P, t_end, rtol, atol, _dev_f64(y_in, (n, mech.n_species)),
                                _dev_f64(y_out, (n, mech.n_species)), _stream_ptr(stream)))
    return y_out


def chem_integrate_ex(mech: Mechanism, P: float, t_end: float, rtol: float, atol: float, y_in, y_out=None,
                      want_stats=True, stream=None, **opts):
    """Hot path with options and per-state statistics.  Returns (y_out, stats) with stats a CUDA uint8 tensor
    of chem_stats records (use stats_to_numpy) or None."""
    import torch
    n = y_in.shape[0]
    if y_out is None:
        y_out = torch.empty_like(y_in)
    stats = torch.zeros((max(n, 1), STATS_DTYPE.itemsize), dtype=torch.uint8, device=y_in.device) if want_stats else None
    o = _opts(**opts)
    _check(lib().chem_integrate_ex(mech._h, n, P, t_end, rtol, atol, _dev_f64(y_in, (n, mech.n_species)),
                                   _dev_f64(y_out, (n, mech.n_species)), C.byref(o),
                                   C.c_void_p(stats.data_ptr()) if want_stats else None, _stream_ptr(stream)))
    return y_out, (stats[:n] if want_stats else None)


NOALLOC_MAX_STATES = 1048576     # CHEM_NOALLOC_MAX_STATES of include/chem.h


def chem_integrate_noalloc(mech: Mechanism, P: float, t_end: float, rtol: float, atol: float, y_in, y_out, stats=None,
                           stream=None, **opts):
    """chem_integrate_ex for callers that may not allocate device memory while they run (an application whose own arena
    holds the whole GPU, a fixed memory budget, a time-critical loop): the library's scratch is a fixed 4 MiB array inside
    libchem.so instead of a per-launch allocation.  This wrapper allocates nothing either: `y_out` [n, N] float64 and the
    optional `stats` (uint8 [n, 48], see stats_to_numpy) are CUDA tensors the caller made beforehand.  At most
    NOALLOC_MAX_STATES states per call (ChemError beyond that), kernel 0, 1 or 2 only, and no two calls may overlap on
    the GPU (they share the array): see include/chem.h.  Returns (y_out, stats)."""
    n = y_in.shape[0]
    o = _opts(**opts)
    if stats is not None and not (stats.is_cuda and stats.is_contiguous() and stats.numel() * stats.element_size() >= n * STATS_DTYPE.itemsize):
        raise ChemError("stats must be a contiguous CUDA tensor of at least n * 48 bytes")
    _check(lib().chem_integrate_noalloc(mech._h, n, P, t_end, rtol, atol, _dev_f64(y_in, (n, mech.n_species)),
                                        _dev_f64(y_out, (n, mech.n_species)), C.byref(o),
                                        C.c_void_p(stats.data_ptr()) if stats is not None else None, _stream_ptr(stream)))
    return y_out, stats


def stats_to_numpy(stats):
    return np.frombuffer(stats.cpu().numpy().tobytes(), dtype=STATS_DTYPE)


def chem_integrate_host(mech: Mechanism, P: float, t_end: float, rtol: float, atol: float, y_in_host: np.ndarray,
                        y_out_host: np.ndarray | None = None, want_stats=False, **opts):
    """End-to-end form with HOST (numpy) buffers; copies are inside the call."""
    y_in_host = np.ascontiguousarray(y_in_host, dtype=np.float64)
    n = y_in_host.shape[0]
    if y_out_host is None:
        y_out_host = np.empty_like(y_in_host)
    stats = np.zeros(n, dtype=STATS_DTYPE) if want_stats else None
    o = _opts(**opts)
    _check(lib().chem_integrate_host(mech._h, n, P, t_end, rtol, atol, C.c_void_p(y_in_host.ctypes.data),
                                     C.c_void_p(y_out_host.ctypes.data), C.byref(o),
                                     C.c_void_p(stats.ctypes.data) if want_stats else None))
    return (y_out_host, stats) if want_stats else y_out_host


KERNEL_NAMES = {0: "none", 1: "integrate_kernel (group per state)", 2: "integrate_warp_kernel (warp per state)",
                3: "integrate_tps_kernel (thread per state)"}


def chem_last_kernel(mech: Mechanism) -> int:
    return int(lib().chem_last_kernel(mech._h))


def chem_fp64_probe(iters: int = 1 << 16, reps: int = 5) -> float:
    """measured fp64 FMA rate of the device in TFLOP/s (diagnostic; include/chem.h)"""
    out = C.c_double(0.0)
    _check(lib().chem_fp64_probe(iters, reps, C.byref(out)))
    return float(out.value)


def chem_scratch_trim() -> None:
    """return the launch scratch cached by the library's memory pool on the current device to the driver"""
    _check(lib().chem_scratch_trim())


def chem_launch_count() -> int:
    return int(lib().chem_launch_count())
