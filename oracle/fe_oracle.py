"""ctypes binding of the CPU oracle (oracle/fe_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It imports nothing from paper_1412_8754_b200's CUDA binding; parameters arrive
as the plain dict made by paper_1412_8754_b200.workloads.model_params.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build


class FeoParams(C.Structure):
    _fields_ = [("model", C.c_int32), ("form_factor", C.c_int32), ("t", C.c_double * 4),
                ("mu", C.c_double), ("U", C.c_double), ("eta_scale", C.c_double),
                ("cond_mult", C.c_double), ("band_mask", C.c_int32), ("const_mode", C.c_int32),
                ("tb3", C.c_double * 13)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int32)
        pp = C.POINTER(FeoParams)
        L.feo_num_bands.argtypes = [pp]
        L.feo_num_bands.restype = C.c_int
        L.feo_num_threads.restype = C.c_int
        L.feo_set_num_threads.argtypes = [C.c_int]
        L.feo_band_energies.argtypes = [pp, C.c_double, C.c_double, dp]
        L.feo_band_energies.restype = None
        L.feo_three_band_matrix.argtypes = [pp, C.c_double, C.c_double, dp, dp]
        L.feo_three_band_matrix.restype = None
        L.feo_herm3_eigvals.argtypes = [dp, dp, dp]
        L.feo_herm3_eigvals.restype = None
        L.feo_eta.argtypes = [pp, C.c_double, C.c_double]
        L.feo_eta.restype = C.c_double
        L.feo_quasiparticle.argtypes = [C.c_double, C.c_double, C.c_double, dp, dp]
        L.feo_quasiparticle.restype = None
        L.feo_thermal.argtypes = [C.c_double, C.c_double]
        L.feo_thermal.restype = C.c_double
        L.feo_omega_column.argtypes = [pp, C.c_int32, C.c_double, C.c_double, C.c_double, C.c_double,
                                       dp, C.c_int32, dp]
        L.feo_omega_column.restype = C.c_int
        L.feo_omega_column_magnitude.argtypes = L.feo_omega_column.argtypes
        L.feo_omega_column_magnitude.restype = C.c_int
        L.feo_omega_grid.argtypes = [pp, C.c_int32, C.c_double, dp, C.c_int32, dp, C.c_int32,
                                     dp, C.c_int32, dp]
        L.feo_omega_grid.restype = C.c_int
        L.feo_argmin.argtypes = [dp, dp, C.c_int32, C.c_int32, ip, dp, dp]
        L.feo_argmin.restype = C.c_int
        L.feo_pair_term.argtypes = [C.c_double, C.c_double, C.c_double]
        L.feo_pair_term.restype = C.c_double
        L.feo_pair_susceptibility.argtypes = [pp, C.c_int32, C.c_double, dp, C.c_int32, C.c_double, dp]
        L.feo_pair_susceptibility.restype = C.c_int
        L.feo_omega_column_sp.argtypes = L.feo_omega_column.argtypes
        L.feo_omega_column_sp.restype = C.c_int
        L.feo_argmin_q.argtypes = [dp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, ip, ip, dp]
        L.feo_argmin_q.restype = C.c_int
        _lib = L
    return _lib


def _params(p: dict) -> FeoParams:
    s = FeoParams()
    s.model, s.form_factor = p["model"], p["form_factor"]
    for i in range(4):
        s.t[i] = p["t"][i]
    s.mu, s.U, s.eta_scale, s.cond_mult = p["mu"], p["U"], p["eta_scale"], p["cond_mult"]
    s.band_mask, s.const_mode = p["band_mask"], p["const_mode"]
    for i, v in enumerate(p.get("tb3", ())):
        s.tb3[i] = v
    return s


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def num_threads() -> int:
    return int(lib().feo_num_threads())


def set_num_threads(n: int) -> None:
    lib().feo_set_num_threads(int(n))


def band_energies(p: dict, kx: float, ky: float) -> np.ndarray:
    sp = _params(p)
    out = np.zeros(3)
    lib().feo_band_energies(C.byref(sp), kx, ky, _dptr(out))
    return out[: {1: 1, 2: 2, 3: 3}[p["model"]]]


def three_band_matrix(p: dict, kx: float, ky: float) -> np.ndarray:
    """Complex 3x3 orbital Hamiltonian T_k of Eqs. B.1-B.6."""
    sp = _params(p)
    re, im = np.zeros(9), np.zeros(9)
    lib().feo_three_band_matrix(C.byref(sp), kx, ky, _dptr(re), _dptr(im))
    return (re + 1j * im).reshape(3, 3)


def herm3_eigvals(a) -> np.ndarray:
    """Ascending eigenvalues of a 3x3 complex Hermitian matrix (the oracle's Jacobi routine)."""
    a = np.asarray(a, dtype=np.complex128).reshape(3, 3)
    re, im = np.ascontiguousarray(a.real).reshape(-1), np.ascontiguousarray(a.imag).reshape(-1)
    out = np.zeros(3)
    lib().feo_herm3_eigvals(_dptr(re), _dptr(im), _dptr(out))
    return out


def eta(p: dict, kx: float, ky: float) -> float:
    sp = _params(p)
    return float(lib().feo_eta(C.byref(sp), kx, ky))


def quasiparticle(a: float, b: float, gap: float):
    ep, em = C.c_double(), C.c_double()
    lib().feo_quasiparticle(a, b, gap, C.byref(ep), C.byref(em))
    return ep.value, em.value


def thermal(x: float, T: float) -> float:
    return float(lib().feo_thermal(x, T))


def omega_column(p: dict, N: int, T: float, q, h: float, delta) -> np.ndarray:
    sp = _params(p)
    d = np.ascontiguousarray(delta, dtype=np.float64)
    out = np.empty(d.shape[0], dtype=np.float64)
    rc = lib().feo_omega_column(C.byref(sp), N, T, float(q[0]), float(q[1]), float(h), _dptr(d), d.shape[0],
                                _dptr(out))
    if rc:
        raise ValueError(f"feo_omega_column failed: {rc}")
    return out


def omega_grid_magnitude(p: dict, N: int, T: float, q, h, delta) -> np.ndarray:
    """Sum of the ABSOLUTE values of the terms of Omega[iq, ih, id] (feo_omega_column_magnitude): the scale the rounding
    of the k-sum acts on; magnitude / |Omega| is the condition number of the sum."""
    sp = _params(p)
    q = np.ascontiguousarray(q, dtype=np.float64).reshape(-1, 2)
    h = np.ascontiguousarray(h, dtype=np.float64).reshape(-1)
    d = np.ascontiguousarray(delta, dtype=np.float64).reshape(-1)
    out = np.empty((q.shape[0], h.shape[0], d.shape[0]), dtype=np.float64)
    for iq in range(q.shape[0]):
        for ih in range(h.shape[0]):
            col = np.empty(d.shape[0], dtype=np.float64)
            rc = lib().feo_omega_column_magnitude(C.byref(sp), N, T, float(q[iq, 0]), float(q[iq, 1]), float(h[ih]),
                                                  _dptr(d), d.shape[0], _dptr(col))
            if rc:
                raise ValueError(f"feo_omega_column_magnitude failed: {rc}")
            out[iq, ih] = col
    return out


def omega_grid(p: dict, N: int, T: float, q, h, delta) -> np.ndarray:
    """Omega[iq, ih, id] over the full grid (Algorithm 1 loop order)."""
    sp = _params(p)
    q = np.ascontiguousarray(q, dtype=np.float64).reshape(-1, 2)
    h = np.ascontiguousarray(h, dtype=np.float64).reshape(-1)
    d = np.ascontiguousarray(delta, dtype=np.float64).reshape(-1)
    out = np.empty((q.shape[0], h.shape[0], d.shape[0]), dtype=np.float64)
    rc = lib().feo_omega_grid(C.byref(sp), N, T, _dptr(q), q.shape[0], _dptr(h), h.shape[0], _dptr(d),
                              d.shape[0], _dptr(out))
    if rc:
        raise ValueError(f"feo_omega_grid failed: {rc}")
    return out


def argmin(omega, delta):
    """Per-(q,h) linear search over the last axis.  Returns (idx int32, delta*, omega*)."""
    om = np.ascontiguousarray(omega, dtype=np.float64)
    d = np.ascontiguousarray(delta, dtype=np.float64).reshape(-1)
    nd = d.shape[0]
    ncol = om.size // nd
    idx = np.empty(ncol, dtype=np.int32)
    ds = np.empty(ncol)
    os_ = np.empty(ncol)
    rc = lib().feo_argmin(_dptr(om), _dptr(d), ncol, nd, idx.ctypes.data_as(C.POINTER(C.c_int32)), _dptr(ds),
                          _dptr(os_))
    if rc:
        raise ValueError(f"feo_argmin failed: {rc}")
    shp = om.shape[:-1]
    return idx.reshape(shp), ds.reshape(shp), os_.reshape(shp)


def argmin_q(omega, ref_id=-1):
    """Per-h global minimum over (q, Delta) of Omega[iq, ih, id] (Algorithm 1 outer loops).
    Returns (iq int32[nh], id int32[nh], value[nh]); value = Omega - Omega[..., ref_id] when ref_id >= 0."""
    om = np.ascontiguousarray(omega, dtype=np.float64)
    nq, nh, nd = om.shape
    iq, idd, val = np.empty(nh, dtype=np.int32), np.empty(nh, dtype=np.int32), np.empty(nh)
    ip = C.POINTER(C.c_int32)
    rc = lib().feo_argmin_q(_dptr(om), nq, nh, nd, int(ref_id), iq.ctypes.data_as(ip), idd.ctypes.data_as(ip), _dptr(val))
    if rc:
        raise ValueError(f"feo_argmin_q failed: {rc}")
    return iq, idd, val


def pair_term(a: float, b: float, T: float) -> float:
    """[f(-a) - f(b)] / (a + b), the thermal factor of Eq. C.3 at omega = 0."""
    return float(lib().feo_pair_term(a, b, T))


def pair_susceptibility(p: dict, N: int, T: float, q, h: float) -> np.ndarray:
    """chi[iq, eps, eps'] of Eqs. C.2-C.3 (static Cooper-pair susceptibility)."""
    sp = _params(p)
    q = np.ascontiguousarray(q, dtype=np.float64).reshape(-1, 2)
    nb = {1: 1, 2: 2, 3: 3}[p["model"]]
    out = np.empty((q.shape[0], nb, nb), dtype=np.float64)
    rc = lib().feo_pair_susceptibility(C.byref(sp), N, T, _dptr(q), q.shape[0], float(h), _dptr(out))
    if rc:
        raise ValueError(f"feo_pair_susceptibility failed: {rc}")
    return out


def omega_grid_sp(p: dict, N: int, T: float, q, h, delta) -> np.ndarray:
    """Omega[iq, ih, id] with every per-term operation in binary32 (the paper's SP build; sum over k in double)."""
    sp = _params(p)
    q = np.ascontiguousarray(q, dtype=np.float64).reshape(-1, 2)
    h = np.ascontiguousarray(h, dtype=np.float64).reshape(-1)
    d = np.ascontiguousarray(delta, dtype=np.float64).reshape(-1)
    out = np.empty((q.shape[0], h.shape[0], d.shape[0]), dtype=np.float64)
    for iq in range(q.shape[0]):
        for ih in range(h.shape[0]):
            col = np.empty(d.shape[0])
            rc = lib().feo_omega_column_sp(C.byref(sp), N, T, float(q[iq, 0]), float(q[iq, 1]), float(h[ih]), _dptr(d),
                                           d.shape[0], _dptr(col))
            if rc:
                raise ValueError(f"feo_omega_column_sp failed: {rc}")
            out[iq, ih] = col
    return out
