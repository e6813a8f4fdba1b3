"""Thin Python binding of libfe (include/fe.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device memory
(`torch.empty(..., device="cuda")`), streams and nothing else.  There is no CPU fallback: if libfe.so is
missing or no B200 is visible, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

FE_OK, FE_EINVAL, FE_ENOMEM, FE_ECUDA, FE_EARCH = 0, -1, -2, -3, -4
EVAL_FACTORED, EVAL_DIRECT, EVAL_WINDOWED, EVAL_COOP, EVAL_COOP_EO = 0, 1, 2, 3, 4

# include/fe.h (the boundary) and include/fe_debug.h (test / tuning hooks)
EXPORTS_API = ["fe_create", "fe_set_temperature", "fe_set_eval_mode", "fe_omega_grid", "fe_argmin", "fe_argmin_q", "fe_pair_susceptibility",
               "fe_omega_grid_sp", "fe_scan_verified", "fe_scan_host", "fe_enable_timing", "fe_get_timing", "fe_get_last_launch_info",
               "fe_get_launch_count", "fe_get_slot_counts", "fe_enable_slot_counts", "fe_omega_grid_static", "fe_static_limits", "fe_set_symmetry", "fe_get_last_symmetry", "fe_fp64_peak_probe", "fe_build_source_hash", "fe_destroy", "fe_strerror"]
EXPORTS_DEBUG = ["fe_set_tuning", "fe_tile_info", "fe_set_debug_flags", "fe_set_coop_shape", "fe_coop_shape_info", "fe_debug_math",
                 "fe_set_chi_table_budget", "fe_debug_sym_index", "fe_debug_coop_occupancy"]
EXPORTS = EXPORTS_API + EXPORTS_DEBUG


class FeError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libfe error {code}: {msg}")
        self.code = code


class ModelParams(C.Structure):
    _fields_ = [("model", C.c_int32), ("form_factor", C.c_int32), ("t", C.c_double * 4),
                ("mu", C.c_double), ("U", C.c_double), ("eta_scale", C.c_double),
                ("cond_mult", C.c_double), ("band_mask", C.c_int32), ("const_mode", C.c_int32),
                ("tb3", C.c_double * 13)]


_lib = None


def lib_path() -> str:
    return _build.LIB


def lib():
    """Load libfe.so (building it in-tree with nvcc if it is missing or stale and nvcc exists)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.stale():
        try:
            _build.build()
        except Exception as e:  # no nvcc on this machine and no prebuilt library: fail loudly
            if not os.path.exists(path):
                raise RuntimeError(f"libfe.so is not built and could not be built here: {e}") from e
    L = C.CDLL(path)
    dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.c_void_p
    L.fe_create.argtypes = [C.POINTER(ModelParams), C.c_int32, C.c_double, C.POINTER(vp)]
    L.fe_set_temperature.argtypes = [vp, C.c_double]
    L.fe_set_eval_mode.argtypes = [vp, C.c_int32]
    L.fe_omega_grid.argtypes = [vp, dp, C.c_int32, dp, C.c_int32, dp, C.c_int32, vp, vp]
    L.fe_argmin.argtypes = [vp, vp, dp, C.c_int32, C.c_int32, vp, vp, vp, vp]
    L.fe_argmin_q.argtypes = [vp, vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, vp, vp, vp]
    L.fe_pair_susceptibility.argtypes = [vp, dp, C.c_int32, C.c_double, vp, vp]
    L.fe_omega_grid_sp.argtypes = [vp, dp, C.c_int32, dp, C.c_int32, dp, C.c_int32, C.c_int32, vp, vp]
    L.fe_scan_verified.argtypes = [vp, dp, C.c_int32, dp, C.c_int32, dp, C.c_int32, C.c_int32, C.c_double, vp, vp, vp,
                                   C.POINTER(C.c_int32), C.POINTER(C.c_int32), vp]
    L.fe_scan_host.argtypes = [vp, dp, C.c_int32, dp, C.c_int32, dp, C.c_int32, vp, vp, vp, vp, vp]
    L.fe_enable_timing.argtypes = [vp, C.c_int32]
    L.fe_get_timing.argtypes = [vp, C.POINTER(C.c_float), dp]
    L.fe_get_launch_count.argtypes = [vp, C.POINTER(C.c_int64)]
    L.fe_get_last_launch_info.argtypes = [vp, ip]
    L.fe_get_slot_counts.argtypes = [vp, dp]
    L.fe_enable_slot_counts.argtypes = [vp, C.c_int32]
    L.fe_debug_sym_index.argtypes = [C.c_int32, C.c_int32, C.c_int64, ip, ip, C.POINTER(C.c_int64)]
    L.fe_debug_coop_occupancy.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_int32, ip]
    L.fe_set_symmetry.argtypes = [vp, C.c_int32]
    L.fe_get_last_symmetry.argtypes = [vp, ip]
    L.fe_set_tuning.argtypes = [vp, C.c_int32, C.c_int32]
    L.fe_tile_info.argtypes = [C.c_int32, ip, ip]
    L.fe_set_debug_flags.argtypes = [vp, C.c_int32]
    L.fe_set_coop_shape.argtypes = [vp, C.c_int32]
    L.fe_set_chi_table_budget.argtypes = [vp, C.c_double]
    L.fe_coop_shape_info.argtypes = [C.c_int32, ip]
    L.fe_fp64_peak_probe.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_float), dp, vp]
    L.fe_debug_math.argtypes = [vp, C.c_int32, C.c_int32, vp, vp, vp]
    L.fe_omega_grid_static.argtypes = [C.POINTER(ModelParams), C.c_int32, C.c_double, dp, C.c_int32, dp, C.c_int32, dp, C.c_int32, vp, vp]
    L.fe_static_limits.argtypes = [C.POINTER(C.c_int64)]
    L.fe_destroy.argtypes = [vp]
    L.fe_destroy.restype = None
    L.fe_strerror.argtypes = [C.c_int]
    L.fe_strerror.restype = C.c_char_p
    L.fe_build_source_hash.argtypes = []
    L.fe_build_source_hash.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("fe_destroy", "fe_strerror", "fe_build_source_hash"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def built_source_hash() -> str:
    """Hash of the kernel sources libfe.so was compiled from (fe_build_source_hash)."""
    return lib().fe_build_source_hash().decode()


def source_hash() -> str:
    """Hash of the kernel sources in the tree now (build.source_hash)."""
    return _build.source_hash()


def _check(rc):
    if rc != FE_OK:
        raise FeError(rc, lib().fe_strerror(rc).decode())


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a.reshape(shape) if shape is not None else a.reshape(-1)


def _stream(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def make_params(p: dict) -> ModelParams:
    s = ModelParams()
    s.model, s.form_factor = p["model"], p["form_factor"]
    for i in range(4):
        s.t[i] = p["t"][i]
    s.mu, s.U, s.eta_scale, s.cond_mult = p["mu"], p["U"], p["eta_scale"], p["cond_mult"]
    s.band_mask, s.const_mode = p["band_mask"], p["const_mode"]
    for i, v in enumerate(p.get("tb3", ())):
        s.tb3[i] = v
    return s


def tiles():
    out, i = [], 1
    th, td = C.c_int32(), C.c_int32()
    while lib().fe_tile_info(i, C.byref(th), C.byref(td)) == FE_OK:
        out.append((th.value, td.value))
        i += 1
    return out


def coop_shapes():
    """[(TH, TD, WH, WD, threads, blocks_per_sm), ...] of the FE_EVAL_COOP shape table (index + 1 = shape id)."""
    out, i = [], 1
    a = (C.c_int32 * 6)()
    while lib().fe_coop_shape_info(i, a) == FE_OK:
        out.append(tuple(a))
        i += 1
    return out


def coop_occupancy(shape, nbands=2, form_factor=1, sym=0):
    """Resident blocks per SM of one cooperative-kernel instance on the current device (fe_debug_coop_occupancy)."""
    v = C.c_int32()
    _check(lib().fe_debug_coop_occupancy(int(shape), int(nbands), int(form_factor), int(sym), C.byref(v)))
    return v.value


def fp64_peak_probe(blocks=148 * 16, iters=1 << 16, stream=None):
    """Measured DFMA rate of the current device: returns (dfma_per_second, ms)."""
    ms, cnt = C.c_float(), C.c_double()
    _check(lib().fe_fp64_peak_probe(blocks, iters, C.byref(ms), C.byref(cnt), _stream(stream)))
    return cnt.value / (ms.value * 1e-3), ms.value


def static_limits():
    """Limits of omega_grid_static (fe_static_limits): dict(list, trig, out, partial, bytes).  No CUDA call."""
    a = (C.c_int64 * 5)()
    _check(lib().fe_static_limits(a))
    return dict(list=a[0], trig=a[1], out=a[2], partial=a[3], bytes=a[4])


def omega_grid_static(params: dict, N: int, T: float, q, h, delta, out, stream=None):
    """Omega[iq, ih, id] on a small grid through fe_omega_grid_static, the entry point for callers that cannot let the
    library allocate: no handle, and all working memory in a fixed array inside libfe.so (limits: static_limits()).

    Nothing is allocated here either, so `out` is required: a contiguous float64 CUDA tensor with nq*nh*nd elements that
    the caller made while it still could.  All calls on a device share the library's one scratch array; keep them on one
    stream (include/fe.h says what happens otherwise).  Returns `out`; asynchronous on `stream` (default: current)."""
    import torch
    q, h, d = _f64(q, (-1, 2)), _f64(h), _f64(delta)
    shape = (q.shape[0], h.shape[0], d.shape[0])
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == int(np.prod(shape))
    p = make_params(params)
    _check(lib().fe_omega_grid_static(C.byref(p), int(N), float(T), _dptr(q), shape[0], _dptr(h), shape[1], _dptr(d), shape[2],
                                      C.c_void_p(out.data_ptr()), _stream(stream)))
    return out


class FreeEnergy:
    """fe_handle wrapper: Omega(Delta; q, h, T) grids and per-(q, h) minima on one B200."""

    def __init__(self, params: dict, N: int, T: float):
        self._h = C.c_void_p()
        self._params = make_params(params)
        self.N, self.T = int(N), float(T)
        self.nbands = {1: 1, 2: 2, 3: 3}[int(params["model"])]
        _check(lib().fe_create(C.byref(self._params), self.N, self.T, C.byref(self._h)))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().fe_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_temperature(self, T):
        _check(lib().fe_set_temperature(self._h, float(T)))
        self.T = float(T)

    def set_eval_mode(self, mode):
        _check(lib().fe_set_eval_mode(self._h, int(mode)))

    def set_tuning(self, tile=0, target_blocks=0):
        _check(lib().fe_set_tuning(self._h, int(tile), int(target_blocks)))

    def set_symmetry(self, on=True):
        """Opt-in mirror-symmetry reduction of the k-sum (fe_set_symmetry)."""
        _check(lib().fe_set_symmetry(self._h, 1 if on else 0))

    def last_symmetry(self):
        """0 none, 1 k_y -> -k_y, 2 k_x -> -k_x, 3 k_x <-> k_y: what the most recent omega_grid launch used."""
        v = C.c_int32()
        _check(lib().fe_get_last_symmetry(self._h, C.byref(v)))
        return v.value

    def set_coop_shape(self, shape=0):
        _check(lib().fe_set_coop_shape(self._h, int(shape)))

    def set_chi_table_budget(self, nbytes):
        _check(lib().fe_set_chi_table_budget(self._h, float(nbytes)))

    def set_debug_flags(self, flags):
        _check(lib().fe_set_debug_flags(self._h, int(flags)))

    def enable_timing(self, on=True):
        _check(lib().fe_enable_timing(self._h, 1 if on else 0))

    def enable_slot_counts(self, on=True):
        """Count slot kinds in the following cooperative launches (atomics in the kernel: keep off while timing)."""
        _check(lib().fe_enable_slot_counts(self._h, 1 if on else 0))

    def last_ksum(self):
        """(ms, band_evals) of the most recent k-sum launch; call after synchronising the stream."""
        ms, be = C.c_float(), C.c_double()
        _check(lib().fe_get_timing(self._h, C.byref(ms), C.byref(be)))
        return ms.value, be.value

    def last_launch_info(self):
        a = (C.c_int32 * 6)()
        _check(lib().fe_get_last_launch_info(self._h, a))
        return dict(th=a[0], td=a[1], ksplit=a[2], grid=a[3], mode=a[4], rows_per_chunk=a[5])

    def slot_counts(self):
        """{dense, a_dominated (= list + series), a_series, b_dominated, padding} slot counts of the most recent cooperative
        k-sum launch made with enable_slot_counts on."""
        a = (C.c_double * 5)()
        _check(lib().fe_get_slot_counts(self._h, a))
        return dict(dense=a[0], a_dominated=a[1] + a[4], a_series=a[4], b_dominated=a[2], padding=a[3])

    def launch_count(self):
        n = C.c_int64()
        _check(lib().fe_get_launch_count(self._h, C.byref(n)))
        return n.value

    def omega_grid(self, q, h, delta, out=None, stream=None):
        """Omega[iq, ih, id] as a CUDA torch tensor (float64).  Asynchronous on `stream` (default: current)."""
        import torch
        q = _f64(q, (-1, 2))
        h = _f64(h)
        d = _f64(delta)
        shape = (q.shape[0], h.shape[0], d.shape[0])
        if out is None:
            out = torch.empty(shape, dtype=torch.float64, device="cuda")
        else:
            assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == int(np.prod(shape))
        _check(lib().fe_omega_grid(self._h, _dptr(q), shape[0], _dptr(h), shape[1], _dptr(d), shape[2],
                                   C.c_void_p(out.data_ptr()), _stream(stream)))
        return out

    def argmin(self, omega, delta, stream=None):
        """(idx int32, delta*, omega*) CUDA tensors of shape omega.shape[:-1]."""
        import torch
        d = _f64(delta)
        nd = d.shape[0]
        assert omega.is_cuda and omega.dtype == torch.float64 and omega.is_contiguous() and omega.shape[-1] == nd
        ncol = omega.numel() // nd
        shp = tuple(omega.shape[:-1])
        idx = torch.empty(shp, dtype=torch.int32, device="cuda")
        ds = torch.empty(shp, dtype=torch.float64, device="cuda")
        os_ = torch.empty(shp, dtype=torch.float64, device="cuda")
        _check(lib().fe_argmin(self._h, C.c_void_p(omega.data_ptr()), _dptr(d), ncol, nd,
                               C.c_void_p(idx.data_ptr()), C.c_void_p(ds.data_ptr()), C.c_void_p(os_.data_ptr()),
                               _stream(stream)))
        return idx, ds, os_

    def argmin_q(self, omega, ref_id=-1, stream=None):
        """Per-h global minimum over (q, Delta) of omega[iq, ih, id]: (iq int32, id int32, value) CUDA tensors [nh]."""
        import torch
        assert omega.is_cuda and omega.dtype == torch.float64 and omega.is_contiguous() and omega.dim() == 3
        nq, nh, nd = omega.shape
        iq = torch.empty(nh, dtype=torch.int32, device="cuda")
        idd = torch.empty(nh, dtype=torch.int32, device="cuda")
        val = torch.empty(nh, dtype=torch.float64, device="cuda")
        _check(lib().fe_argmin_q(self._h, C.c_void_p(omega.data_ptr()), nq, nh, nd, int(ref_id),
                                 C.c_void_p(iq.data_ptr()), C.c_void_p(idd.data_ptr()), C.c_void_p(val.data_ptr()),
                                 _stream(stream)))
        return iq, idd, val

    def pair_susceptibility(self, q, hz, out=None, stream=None):
        """chi[iq, e, f] (Appendix C) as a CUDA torch tensor (float64).  Asynchronous on `stream`."""
        import torch
        q = _f64(q).reshape(-1, 2)
        nb = self.nbands
        if out is None:
            out = torch.empty((q.shape[0], nb, nb), dtype=torch.float64, device="cuda")
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == q.shape[0] * nb * nb
        _check(lib().fe_pair_susceptibility(self._h, _dptr(q), q.shape[0], C.c_double(float(hz)),
                                            C.c_void_p(out.data_ptr()), _stream(stream)))
        return out

    def omega_grid_sp(self, q, h, delta, fast_math=False, out=None, stream=None):
        """Omega[iq, ih, id] from the single-precision kernels (the paper's SP / SPFM builds), as float64 tensor."""
        import torch
        q, h, d = _f64(q).reshape(-1, 2), _f64(h), _f64(delta)
        if out is None:
            out = torch.empty((q.shape[0], h.shape[0], d.shape[0]), dtype=torch.float64, device="cuda")
        _check(lib().fe_omega_grid_sp(self._h, _dptr(q), q.shape[0], _dptr(h), h.shape[0], _dptr(d), d.shape[0],
                                      int(bool(fast_math)), C.c_void_p(out.data_ptr()), _stream(stream)))
        return out

    def scan_verified(self, q, h, delta, fast_math=False, margin_rel=1e-5, stream=None, screen=None):
        """Low-precision screening + fp64 verification of the candidates: (idx, delta*, omega*, n_verified, n_changed);
        n_changed = columns whose minimum the fp64 verification moved away from the single-precision argmin.
        screen: "sp" | "spfm" (the paper's single-precision builds) -- overrides fast_math when given."""
        import torch
        if screen is not None:
            fast_math = {"sp": 0, "spfm": 1}[screen]
        q, h, d = _f64(q).reshape(-1, 2), _f64(h), _f64(delta)
        shp = (q.shape[0], h.shape[0])
        idx = torch.empty(shp, dtype=torch.int32, device="cuda")
        ds = torch.empty(shp, dtype=torch.float64, device="cuda")
        os_ = torch.empty(shp, dtype=torch.float64, device="cuda")
        nv, nc = C.c_int32(0), C.c_int32(0)
        _check(lib().fe_scan_verified(self._h, _dptr(q), q.shape[0], _dptr(h), h.shape[0], _dptr(d), d.shape[0],
                                      int(bool(fast_math)), float(margin_rel), C.c_void_p(idx.data_ptr()),
                                      C.c_void_p(ds.data_ptr()), C.c_void_p(os_.data_ptr()), C.byref(nv), C.byref(nc),
                                      _stream(stream)))
        return idx, ds, os_, nv.value, nc.value

    def scan_host(self, q, h, delta, want_omega=True, out=None, stream=None):
        """Host-buffer end-to-end path (fe_scan_host): numpy in, numpy out, synchronous.

        `out` may carry preallocated (pinned) numpy views: dict with keys omega/idx/delta_star/omega_star."""
        q = _f64(q, (-1, 2))
        h = _f64(h)
        d = _f64(delta)
        nq, nh, nd = q.shape[0], h.shape[0], d.shape[0]
        out = out or {}
        om = out.get("omega") if want_omega else None
        if want_omega and om is None:
            om = np.empty((nq, nh, nd), dtype=np.float64)
        idx = out.get("idx", None)
        idx = np.empty((nq, nh), dtype=np.int32) if idx is None else idx
        ds = out.get("delta_star", None)
        ds = np.empty((nq, nh), dtype=np.float64) if ds is None else ds
        os_ = out.get("omega_star", None)
        os_ = np.empty((nq, nh), dtype=np.float64) if os_ is None else os_
        _check(lib().fe_scan_host(self._h, _dptr(q), nq, _dptr(h), nh, _dptr(d), nd,
                                  C.c_void_p(om.ctypes.data) if om is not None else None,
                                  C.c_void_p(idx.ctypes.data), C.c_void_p(ds.ctypes.data), C.c_void_p(os_.ctypes.data),
                                  _stream(stream)))
        return om, idx, ds, os_

    def debug_math(self, which, x):
        import torch
        assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
        y = torch.empty_like(x)
        _check(lib().fe_debug_math(self._h, int(which), x.numel(), C.c_void_p(x.data_ptr()), C.c_void_p(y.data_ptr()),
                                   _stream(None)))
        return y
