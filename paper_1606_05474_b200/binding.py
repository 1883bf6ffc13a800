"""Thin ctypes binding of include/helios.h (argument marshalling only).

PyTorch supplies device memory and the stream; every step of the path runs inside
libhelios_b200.so.  There is no CPU fallback: if the library cannot be loaded or no CUDA device
is present the calls raise HeliosError.  Names mirror the C-ABI (helios_setup / helios_fluxes /
helios_iterate_re ...).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

OK, E_BADARG, E_NOTSETUP, E_CUDA, E_NONFINITE, E_WORKSPACE = 0, -1, -2, -3, -4, -5
PREC_FP64, PREC_FP32 = 0, 1
NSCAT_DIRECT = -1   # HELIOS_NSCAT_DIRECT: n_scat value selecting the direct coupled solve

EXPORTS = ["helios_workspace_bytes", "helios_setup", "helios_set_columns", "helios_set_columns_host",
           "helios_set_temperatures", "helios_set_scattering", "helios_fluxes", "helios_fluxes_static", "helios_fluxes_host", "helios_iterate_re",
           "helios_iterate_re_host", "helios_get_re_state", "helios_get_re_metrics", "helios_set_re_state", "helios_get_fluxes",
           "helios_enable_timing", "helios_kernel_time_ms", "helios_launch_count", "helios_launch_shape", "helios_measure_fma_peak", "helios_measure_fma3_peak",
           "helios_last_error", "helios_destroy"]


class HeliosError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"helios error {code}: {msg}")
        self.code = code


class HeliosParams(C.Structure):
    _fields_ = [("n_cols", C.c_int32), ("n_layers", C.c_int32), ("n_bins", C.c_int32),
                ("n_g", C.c_int32), ("ntab_p", C.c_int32), ("ntab_t", C.c_int32),
                ("precision", C.c_int32), ("n_scat", C.c_int32), ("warm_start", C.c_int32),
                ("isothermal_layers", C.c_int32), ("D", C.c_double), ("gravity", C.c_double),
                ("dtau_iso", C.c_double), ("one_minus_w0_min", C.c_double),
                ("dT_frac_max", C.c_double), ("T_floor", C.c_double), ("flux_floor", C.c_double),
                ("exact_absorption", C.c_int32), ("planck_table_dT", C.c_double),
                ("planck_table_Tmax", C.c_double), ("trans_table_dlog10k", C.c_double)]


_lib = None
_VP = C.c_void_p


def lib_path() -> str:
    return _build.LIB


def load():
    """Loads (building first if stale) the C-ABI library.  Raises if it cannot be built/loaded."""
    global _lib
    if _lib is None:
        path = _build.build(accept_dev=True)
        L = C.CDLL(path)
        L.helios_workspace_bytes.restype = C.c_size_t
        L.helios_workspace_bytes.argtypes = [C.POINTER(HeliosParams)]
        L.helios_setup.restype = C.c_int
        L.helios_setup.argtypes = [C.POINTER(_VP), C.POINTER(HeliosParams)] + [_VP] * 10 + [_VP, C.c_size_t, _VP]
        L.helios_set_columns.restype = C.c_int
        L.helios_set_columns.argtypes = [_VP] * 6
        L.helios_set_columns_host.restype = C.c_int
        L.helios_set_columns_host.argtypes = [_VP] * 6
        L.helios_set_temperatures.restype = C.c_int
        L.helios_set_temperatures.argtypes = [_VP, _VP]
        L.helios_set_scattering.restype = C.c_int
        L.helios_set_scattering.argtypes = [_VP, _VP]
        L.helios_fluxes.restype = C.c_int
        L.helios_fluxes.argtypes = [_VP] * 5
        L.helios_fluxes_static.restype = C.c_int
        L.helios_fluxes_static.argtypes = [_VP] * 3
        L.helios_fluxes_host.restype = C.c_int
        L.helios_fluxes_host.argtypes = [_VP] * 4
        L.helios_iterate_re.restype = C.c_int
        L.helios_iterate_re.argtypes = [_VP, C.c_int32, C.c_double, C.c_double, C.c_int32, _VP, _VP, _VP]
        L.helios_iterate_re_host.restype = C.c_int
        L.helios_iterate_re_host.argtypes = [_VP, C.c_int32, C.c_double, C.c_double, C.c_int32, _VP, _VP, _VP]
        L.helios_get_re_state.restype = C.c_int
        L.helios_get_re_state.argtypes = [_VP] * 4
        L.helios_get_re_metrics.restype = C.c_int
        L.helios_get_re_metrics.argtypes = [_VP] * 4
        L.helios_set_re_state.restype = C.c_int
        L.helios_set_re_state.argtypes = [_VP] * 5
        L.helios_get_fluxes.restype = C.c_int
        L.helios_get_fluxes.argtypes = [_VP] * 3
        L.helios_enable_timing.restype = C.c_int
        L.helios_enable_timing.argtypes = [_VP, C.c_int32]
        L.helios_kernel_time_ms.restype = C.c_int
        L.helios_kernel_time_ms.argtypes = [_VP, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.helios_launch_count.restype = C.c_int64
        L.helios_launch_count.argtypes = [_VP]
        L.helios_launch_shape.restype = C.c_int
        L.helios_launch_shape.argtypes = [_VP, C.POINTER(C.c_int32)]
        L.helios_measure_fma_peak.restype = C.c_double
        L.helios_measure_fma_peak.argtypes = [C.c_int32, _VP]
        L.helios_measure_fma3_peak.restype = C.c_double
        L.helios_measure_fma3_peak.argtypes = [C.c_int32, _VP]
        L.helios_last_error.restype = C.c_char_p
        L.helios_last_error.argtypes = [_VP]
        L.helios_destroy.restype = None
        L.helios_destroy.argtypes = [_VP]
        _lib = L
    return _lib


def params_from_dict(d: dict) -> HeliosParams:
    opt = {"flux_floor": 0.0, "exact_absorption": 0, "planck_table_dT": 0.0, "planck_table_Tmax": 0.0,
           "trans_table_dlog10k": 0.0}
    return HeliosParams(**{k: (d.get(k, opt[k]) if k in opt else d[k]) for k, _ in HeliosParams._fields_})


def helios_workspace_bytes(params: dict) -> int:
    p = params_from_dict(params)
    return int(load().helios_workspace_bytes(C.byref(p)))


def helios_measure_fma_peak(precision: int = PREC_FP64, stream: int = 0) -> float:
    return float(load().helios_measure_fma_peak(int(precision), _VP(stream)))


def helios_measure_fma3_peak(precision: int = PREC_FP64, stream: int = 0) -> float:
    return float(load().helios_measure_fma3_peak(int(precision), _VP(stream)))


def _ptr(t):
    return _VP(0) if t is None else _VP(t.data_ptr())


def _hptr(a):
    return _VP(0) if a is None else _VP(a.ctypes.data)


class Helios:
    """One context of the C-ABI library on the current CUDA device.

    `inp` is a paper_1606_05474_b200.inputs.HeliosInputs (numpy arrays); they are uploaded once
    with torch and handed to helios_setup / helios_set_columns as device pointers.
    """

    def __init__(self, inp, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise HeliosError(E_CUDA, "no CUDA device (there is no CPU fallback)")
        self.torch = torch
        self.L = load()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.params = dict(inp.params)
        self.nc, self.n = self.params["n_cols"], self.params["n_layers"]
        self.nb, self.ng = self.params["n_bins"], self.params["n_g"]
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._p = params_from_dict(self.params)
        nbytes = int(self.L.helios_workspace_bytes(C.byref(self._p)))
        if nbytes == 0:
            raise HeliosError(E_BADARG, "invalid parameters")
        up = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(self.device)
        with torch.cuda.stream(self.stream):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self.d = {k: up(getattr(inp, k)) for k in
                      ("p_layer", "p_interface", "bin_edges", "g_pts", "g_wts", "ktab", "tab_log10p",
                       "tab_t", "w0", "g0")}
        ws_ptr = (self.workspace.data_ptr() + 255) // 256 * 256
        self.ctx = _VP()
        r = self.L.helios_setup(C.byref(self.ctx), C.byref(self._p),
                                *[_ptr(self.d[k]) for k in ("p_layer", "p_interface", "bin_edges", "g_pts",
                                                            "g_wts", "ktab", "tab_log10p", "tab_t", "w0", "g0")],
                                _VP(ws_ptr), C.c_size_t(nbytes), _VP(self.stream.cuda_stream))
        if r != OK:
            raise HeliosError(r, self.L.helios_last_error(_VP(0)).decode())
        self.cols = None
        if inp.T0 is not None:
            self.helios_set_columns(inp.T0, inp.f_star, inp.f_star_scale, inp.t_intern, inp.kscale)
        if getattr(inp, "kappa_scat", None) is not None:
            self.helios_set_scattering(inp.kappa_scat)

    # -- helpers ------------------------------------------------------------------------------
    def _check(self, r):
        if r != OK:
            raise HeliosError(r, self.L.helios_last_error(self.ctx).decode())

    def _dev(self, a):
        torch = self.torch
        if a is None:
            return None
        if isinstance(a, torch.Tensor):
            return a.to(device=self.device, dtype=torch.float64).contiguous()
        return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(self.device)

    def empty(self, *shape, dtype=None):
        return self.torch.empty(*shape, dtype=dtype or self.torch.float64, device=self.device)

    # -- C-ABI calls --------------------------------------------------------------------------
    def helios_set_columns(self, T, f_star, f_star_scale, t_intern, kscale):
        with self.torch.cuda.stream(self.stream):
            self.cols = [self._dev(x) for x in (T, f_star, f_star_scale, t_intern, kscale)]
        self._check(self.L.helios_set_columns(self.ctx, *[_ptr(x) for x in self.cols]))

    def helios_set_columns_host(self, T, f_star, f_star_scale, t_intern, kscale):
        arrs = [None if x is None else np.ascontiguousarray(x, dtype=np.float64)
                for x in (T, f_star, f_star_scale, t_intern, kscale)]
        self._check(self.L.helios_set_columns_host(self.ctx, *[_hptr(x) for x in arrs]))

    def helios_set_scattering(self, kappa_scat):
        with self.torch.cuda.stream(self.stream):
            k = self._dev(kappa_scat)
        self._check(self.L.helios_set_scattering(self.ctx, _ptr(k)))
        self._keep_kscat = k

    def helios_set_temperatures(self, T):
        with self.torch.cuda.stream(self.stream):
            t = self._dev(T)
        self._check(self.L.helios_set_temperatures(self.ctx, _ptr(t)))
        self._keep = t

    def helios_fluxes(self, want_spectra=False, out=None):
        """Returns device tensors (F_up, F_dn[, spec_up_toa, spec_dn_boa]); asynchronous."""
        with self.torch.cuda.stream(self.stream):
            F_up, F_dn = out if out is not None else (self.empty(self.nc, self.n + 1), self.empty(self.nc, self.n + 1))
            su = self.empty(self.nc, self.nb) if want_spectra else None
            sd = self.empty(self.nc, self.nb) if want_spectra else None
        self._check(self.L.helios_fluxes(self.ctx, _ptr(F_up), _ptr(F_dn), _ptr(su), _ptr(sd)))
        return (F_up, F_dn, su, sd) if want_spectra else (F_up, F_dn)

    def helios_fluxes_static(self, out):
        """helios_fluxes without any allocation inside the call (scratch in the library's static device array):
        `out` = (F_up, F_dn) device tensors [nc][n+1] the caller already holds; asynchronous."""
        F_up, F_dn = out
        self._check(self.L.helios_fluxes_static(self.ctx, _ptr(F_up), _ptr(F_dn)))
        return F_up, F_dn

    def helios_fluxes_host(self, T_host, F_up_host, F_dn_host):
        """Host numpy buffers in and out; copies happen inside the C call; synchronous."""
        self._check(self.L.helios_fluxes_host(self.ctx, _hptr(T_host), _hptr(F_up_host), _hptr(F_dn_host)))

    def helios_iterate_re(self, max_iter, tol_dT=0.0, tol_flux=0.0, poll_every=0):
        """Returns device tensors dict(T, iters, converged)."""
        torch = self.torch
        with torch.cuda.stream(self.stream):
            T = self.empty(self.nc, self.n)
            iters = self.empty(self.nc, dtype=torch.int32)
            conv = self.empty(self.nc, dtype=torch.int32)
        self._check(self.L.helios_iterate_re(self.ctx, int(max_iter), float(tol_dT), float(tol_flux),
                                             int(poll_every), _ptr(T), _ptr(iters), _ptr(conv)))
        return dict(T=T, iters=iters, converged=conv)

    def helios_iterate_re_host(self, max_iter, T_host_inout, iters_host, converged_host,
                               tol_dT=0.0, tol_flux=0.0, poll_every=0):
        self._check(self.L.helios_iterate_re_host(self.ctx, int(max_iter), float(tol_dT), float(tol_flux),
                                                  int(poll_every), _hptr(T_host_inout), _hptr(iters_host),
                                                  _hptr(converged_host)))

    def helios_get_re_state(self):
        torch = self.torch
        with torch.cuda.stream(self.stream):
            a = self.empty(self.nc, self.n)
            h = self.empty(self.nc, self.n, dtype=torch.int32)
            dT = self.empty(self.nc, self.n)
        self._check(self.L.helios_get_re_state(self.ctx, _ptr(a), _ptr(h), _ptr(dT)))
        return dict(step_factor=a, sign_hist=h, dT_last=dT)

    def helios_get_re_metrics(self):
        torch = self.torch
        with torch.cuda.stream(self.stream):
            m = self.empty(self.nc)
            r = self.empty(self.nc)
            nf = self.empty(self.nc, dtype=torch.int32)
        self._check(self.L.helios_get_re_metrics(self.ctx, _ptr(m), _ptr(r), _ptr(nf)))
        return dict(max_dT=m, max_rel_dF=r, nonfinite=nf)

    def helios_set_re_state(self, step_factor=None, sign_hist=None, iters=None, converged=None):
        torch = self.torch
        with torch.cuda.stream(self.stream):
            a = self._dev(step_factor)
            i32 = lambda x: None if x is None else torch.as_tensor(np.ascontiguousarray(x, dtype=np.int32)).to(self.device)
            h, it, cv = i32(sign_hist), i32(iters), i32(converged)
        self._check(self.L.helios_set_re_state(self.ctx, _ptr(a), _ptr(h), _ptr(it), _ptr(cv)))
        self._keep_state = (a, h, it, cv)

    def helios_get_fluxes(self):
        with self.torch.cuda.stream(self.stream):
            F_up, F_dn = self.empty(self.nc, self.n + 1), self.empty(self.nc, self.n + 1)
        self._check(self.L.helios_get_fluxes(self.ctx, _ptr(F_up), _ptr(F_dn)))
        return F_up, F_dn

    def helios_enable_timing(self, on=True):
        self._check(self.L.helios_enable_timing(self.ctx, 1 if on else 0))

    def helios_kernel_time_ms(self):
        ms, cnt = C.c_double(), C.c_int64()
        self._check(self.L.helios_kernel_time_ms(self.ctx, C.byref(ms), C.byref(cnt)))
        return ms.value, cnt.value

    def helios_launch_count(self) -> int:
        return int(self.L.helios_launch_count(self.ctx))

    def helios_launch_shape(self):
        out = (C.c_int32 * 5)()
        self._check(self.L.helios_launch_shape(self.ctx, out))
        return dict(grid_x=out[0], grid_y=out[1], threads=out[2], smem=out[3], S=out[4])

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        if self.ctx:
            self.stream.synchronize()
            self.L.helios_destroy(self.ctx)
            self.ctx = _VP()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
