"""ctypes binding of oracle/helios_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It builds liboracle.so with gcc on first use (building the checker is not
using it) and marshals numpy arrays; it holds no arithmetic of the method (diffusivity_sweep, the experiment of
PAPER.md section 3.1.5, only loops over the C routines and takes differences of what they return).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "helios_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


class OrcParams(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_bins", C.c_int32), ("n_g", C.c_int32),
                ("ntab_p", C.c_int32), ("ntab_t", C.c_int32), ("n_scat", C.c_int32),
                ("warm_start", C.c_int32), ("isothermal_layers", C.c_int32),
                ("D", C.c_double), ("gravity", C.c_double), ("dtau_iso", C.c_double),
                ("one_minus_w0_min", C.c_double), ("dT_frac_max", C.c_double),
                ("T_floor", C.c_double), ("flux_floor", C.c_double), ("exact_absorption", C.c_int32),
                ("planck_table_dT", C.c_double), ("planck_table_Tmax", C.c_double),
                ("trans_table_dlog10k", C.c_double)]


class OrcCoeffs(C.Structure):
    _fields_ = [("branch", C.c_int32), ("pad_", C.c_int32), ("trans", C.c_double),
                ("alpha", C.c_double), ("beta", C.c_double), ("xi", C.c_double),
                ("S_up", C.c_double), ("S_dn", C.c_double), ("x", C.c_double)]


_D = C.c_double
_I = C.c_int
_PD = C.POINTER(C.c_double)
_PI32 = C.POINTER(C.c_int32)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_num_threads.restype = _I
        L.orc_sigma_sb.restype = _D
        for name, args in [("orc_planck_G_upper", [_D]), ("orc_planck_H_lower", [_D]),
                           ("orc_planck_integral", [_D, _D]), ("orc_planck_bin_mean", [_D, _D, _D]),
                           ("orc_sublayer_dtau", [_D] * 5),
                           ("orc_exact_transmissivity_quadrature", [_D, _I]),
                           ("orc_expint_E1", [_D]), ("orc_exact_transmissivity", [_D]),
                           ("orc_planck_bin_mean_tabulated", [_D] * 4),
                           ("orc_transmission_tabulated", [_D] * 3),
                           ("orc_re_delta_T", [_D] * 6)]:
            f = getattr(L, name)
            f.restype = _D
            f.argtypes = args
        L.orc_kappa_interp.restype = _D
        L.orc_kappa_interp.argtypes = [_PD, _I, _I, _I, _I, _PD, _PD, _D, _D, _I, _I]
        L.orc_level_pressures.argtypes = [_I, _PD, _PD, _PD]
        L.orc_level_temperatures.argtypes = [_I, _PD, _PD, _PD, _PD]
        L.orc_sublayer_coeffs.argtypes = [_D] * 8 + [C.POINTER(OrcCoeffs)]
        L.orc_ray_fluxes.argtypes = [_I, _PD, _PD, _PD] + [_D] * 7 + [_I, _I, _PD, _PD]
        L.orc_exact_layer_eq4.argtypes = [_D] * 6 + [_PD, _PD]
        L.orc_ray_fluxes_w0s.argtypes = [_I, _PD, _PD, _PD, _PD] + [_D] * 6 + [_I, _I, _PD, _PD]
        L.orc_ray_fluxes_exact.argtypes = [_I, _PD, _PD, _PD, _D, _D, _D, _PD, _PD]
        L.orc_fluxes_batch.argtypes = [C.POINTER(OrcParams), _I] + [_PD] * 19
        L.orc_iterate_re.argtypes = ([C.POINTER(OrcParams), _I] + [_PD] * 15 + [_I, _D, _D]
                                     + [_PD, _PI32, _PI32, _PI32, _PD, _PD])
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_PD)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def params_from_dict(d: dict) -> OrcParams:
    opt = {"flux_floor": 0.0, "exact_absorption": 0, "planck_table_dT": 0.0, "planck_table_Tmax": 0.0,
           "trans_table_dlog10k": 0.0}
    return OrcParams(**{k: d.get(k, opt[k]) if k in opt else d[k] for k, _ in OrcParams._fields_})


def num_threads() -> int:
    return int(lib().orc_num_threads())


def sigma_sb() -> float:
    return float(lib().orc_sigma_sb())


def planck_bin_mean(nu_lo, nu_hi, T) -> float:
    return float(lib().orc_planck_bin_mean(float(nu_lo), float(nu_hi), float(T)))


def kappa_interp(ktab, tab_log10p, tab_t, P, T, bin_, g) -> float:
    ktab = _f64(ktab)
    ntp, ntt, nb, ng = ktab.shape
    return float(lib().orc_kappa_interp(_p(ktab), ntp, ntt, nb, ng, _p(_f64(tab_log10p)),
                                        _p(_f64(tab_t)), float(P), float(T), int(bin_), int(g)))


def level_temperatures(p_layer, p_interface, T):
    p_layer, p_interface, T = _f64(p_layer), _f64(p_interface), _f64(T)
    n = T.size
    out = np.empty(2 * n + 1)
    lib().orc_level_temperatures(n, _p(p_layer), _p(p_interface), _p(T), _p(out))
    return out


def level_pressures(p_layer, p_interface):
    p_layer, p_interface = _f64(p_layer), _f64(p_interface)
    n = p_layer.size
    out = np.empty(2 * n + 1)
    lib().orc_level_pressures(n, _p(p_layer), _p(p_interface), _p(out))
    return out


def sublayer_coeffs(dtau, w0, g0, D, B_lo, B_up, dtau_iso=1e-4, omw_min=1e-6) -> OrcCoeffs:
    c = OrcCoeffs()
    lib().orc_sublayer_coeffs(dtau, w0, g0, D, B_lo, B_up, dtau_iso, omw_min, C.byref(c))
    return c


def ray_fluxes(dtau, B_lo, B_up, w0, g0, D, F_dn_top, piB_intern, n_sweeps,
               dtau_iso=1e-4, omw_min=1e-6, F_up_warm=None):
    dtau, B_lo, B_up = _f64(dtau), _f64(B_lo), _f64(B_up)
    nsub = dtau.size
    F_up = np.zeros(nsub + 1) if F_up_warm is None else _f64(F_up_warm).copy()
    F_dn = np.zeros(nsub + 1)
    lib().orc_ray_fluxes(nsub, _p(dtau), _p(B_lo), _p(B_up), w0, g0, D, dtau_iso, omw_min,
                         F_dn_top, piB_intern, int(n_sweeps), 0 if F_up_warm is None else 1,
                         _p(F_up), _p(F_dn))
    return F_up, F_dn


def ray_fluxes_w0s(dtau, B_lo, B_up, w0s, g0, D, F_dn_top, piB_intern, n_sweeps, dtau_iso=1e-4, omw_min=1e-6):
    dtau, B_lo, B_up, w0s = _f64(dtau), _f64(B_lo), _f64(B_up), _f64(w0s)
    nsub = dtau.size
    F_up, F_dn = np.zeros(nsub + 1), np.zeros(nsub + 1)
    lib().orc_ray_fluxes_w0s(nsub, _p(dtau), _p(B_lo), _p(B_up), _p(w0s), g0, D, dtau_iso, omw_min,
                             F_dn_top, piB_intern, int(n_sweeps), 0, _p(F_up), _p(F_dn))
    return F_up, F_dn


def ray_fluxes_exact(dtau, B_lo, B_up, F_dn_top, piB_intern, dtau_iso=1e-4):
    dtau, B_lo, B_up = _f64(dtau), _f64(B_lo), _f64(B_up)
    nsub = dtau.size
    F_up, F_dn = np.zeros(nsub + 1), np.zeros(nsub + 1)
    lib().orc_ray_fluxes_exact(nsub, _p(dtau), _p(B_lo), _p(B_up), dtau_iso, F_dn_top, piB_intern, _p(F_up), _p(F_dn))
    return F_up, F_dn


def exact_layer_eq4(dtau, trans, B_lo, B_up, F_up_lo, F_dn_up):
    a, b = C.c_double(), C.c_double()
    lib().orc_exact_layer_eq4(dtau, trans, B_lo, B_up, F_up_lo, F_dn_up, C.byref(a), C.byref(b))
    return a.value, b.value


def fluxes(inp, T=None, want_spectra=False):
    """Bolometric interface fluxes of every column of `inp` (a HeliosInputs-like object)."""
    p = params_from_dict(inp.params)
    nc, n, nb = inp.params["n_cols"], inp.params["n_layers"], inp.params["n_bins"]
    T = _f64(inp.T0 if T is None else T).reshape(nc, n)
    F_up = np.empty((nc, n + 1))
    F_dn = np.empty((nc, n + 1))
    su = np.empty((nc, nb)) if want_spectra else None
    sd = np.empty((nc, nb)) if want_spectra else None
    arrs = [_f64(a) for a in (inp.p_layer, inp.p_interface, inp.bin_edges, inp.g_wts, inp.ktab,
                              inp.tab_log10p, inp.tab_t, inp.w0, inp.g0)]
    arrs.append(None if getattr(inp, "kappa_scat", None) is None else _f64(inp.kappa_scat))
    fs, fsc, ti, ks = _f64(inp.f_star), _f64(inp.f_star_scale), _f64(inp.t_intern), _f64(inp.kscale)
    lib().orc_fluxes_batch(C.byref(p), nc, *[_p(a) for a in arrs], _p(T), _p(fs), _p(fsc), _p(ti),
                           _p(ks), _p(F_up), _p(F_dn), _p(su), _p(sd))
    if want_spectra:
        return F_up, F_dn, su, sd
    return F_up, F_dn


def iterate_re(inp, max_iter, tol_dT=0.0, tol_flux=0.0, T=None, state=None):
    """Runs the RE iteration; returns dict(T, iters, converged, step_factor, sign_hist, dT_last).
    `state` = a previous return value to chain calls."""
    p = params_from_dict(inp.params)
    nc, n, nb, ng = (inp.params[k] for k in ("n_cols", "n_layers", "n_bins", "n_g"))
    if state is None:
        Tc = _f64(inp.T0 if T is None else T).reshape(nc, n).copy()
        a = np.ones((nc, n))
        h = np.zeros((nc, n), dtype=np.int32)
        iters = np.zeros(nc, dtype=np.int32)
        conv = np.zeros(nc, dtype=np.int32)
        fup = None
        if inp.params["warm_start"]:
            nlev = (n if inp.params["isothermal_layers"] else 2 * n) + 1
            fup = np.zeros((nc, nb, ng, nlev))
    else:
        Tc, a, h = state["T"].copy(), state["step_factor"].copy(), state["sign_hist"].copy()
        iters, conv, fup = state["iters"].copy(), state["converged"].copy(), state.get("fup")
    dT_last = np.zeros((nc, n))
    arrs = [_f64(x) for x in (inp.p_layer, inp.p_interface, inp.bin_edges, inp.g_wts, inp.ktab,
                              inp.tab_log10p, inp.tab_t, inp.w0, inp.g0)]
    arrs.append(None if getattr(inp, "kappa_scat", None) is None else _f64(inp.kappa_scat))
    fs, fsc, ti, ks = _f64(inp.f_star), _f64(inp.f_star_scale), _f64(inp.t_intern), _f64(inp.kscale)
    lib().orc_iterate_re(C.byref(p), nc, *[_p(x) for x in arrs], _p(Tc), _p(fs), _p(fsc), _p(ti),
                         _p(ks), int(max_iter), float(tol_dT), float(tol_flux), _p(a),
                         h.ctypes.data_as(_PI32), iters.ctypes.data_as(_PI32),
                         conv.ctypes.data_as(_PI32), _p(dT_last), _p(fup))
    return dict(T=Tc, iters=iters, converged=conv, step_factor=a, sign_hist=h, dT_last=dT_last,
                fup=fup)


def diffusivity_sweep(inp, D_values=(1.66, 1.8, 1.9, 2.0), max_iter=20000, tol_dT=1.0e-3):
    """Section 3.1.5 of the paper (Fig. 11) with the oracle: a purely absorbing column iterated to
    radiative equilibrium with the exact solver (eq. 3-6) and with the two-stream solver for each D; returns
    {"exact": run, D: run} where run = dict(T, iters, converged, spectrum) and the two-stream runs also hold their
    deviation from the exact run (dT_max, dT_rms [K]; spec_mean, spec_max relative, floor 1e-3 of the brightest bin)."""
    import dataclasses
    nb = inp.params["n_bins"]

    def run(**params):
        i2 = dataclasses.replace(inp, w0=np.zeros(nb), g0=np.zeros(nb), kappa_scat=None,
                                 params=dict(inp.params, n_scat=0, **params))
        st = iterate_re(i2, max_iter, tol_dT=tol_dT)
        spec = fluxes(i2, T=st["T"], want_spectra=True)[2]
        return dict(T=st["T"], iters=st["iters"], converged=st["converged"], spectrum=spec)

    res = {"exact": run(exact_absorption=1)}
    ex = res["exact"]
    floor = 1.0e-3 * np.max(ex["spectrum"], axis=1, keepdims=True)
    for D in D_values:
        r = run(exact_absorption=0, D=float(D))
        dT = r["T"] - ex["T"]
        ds = np.abs(r["spectrum"] - ex["spectrum"]) / np.maximum(ex["spectrum"], floor)
        r.update(dT_max=float(np.max(np.abs(dT))), dT_rms=float(np.sqrt(np.mean(dT * dT))),
                 spec_mean=float(np.mean(ds)), spec_max=float(np.max(ds)))
        res[float(D)] = r
    return res


def scattering_trends(inp, w0=0.5, g0_values=(-0.5, 0.0, 0.5), split_um=1.0, max_iter=20000, tol_dT=1.0e-3):
    """Section 3.1.2 of the paper (Fig. 8) with the oracle: the column iterated to radiative
    equilibrium as a pure absorber and with w0 "across all wavelengths" for each g0, coupled system solved (n_scat = -1);
    returns {"absorption": run, g0: run} with run = dict(T, iters, converged, spectrum, reflected, thermal): the TOA
    emission spectrum at the converged profile and its integrals below / above split_um (the paper's "reflected light
    at <~ 1 um" and "thermal emission at >~ 1 um")."""
    import dataclasses
    nb = inp.params["n_bins"]
    lam_um = 1.0e4 / (0.5 * (inp.bin_edges[:-1] + inp.bin_edges[1:]))
    dnu = np.diff(inp.bin_edges)

    def run(w, g):
        i2 = dataclasses.replace(inp, w0=np.full(nb, float(w)), g0=np.full(nb, float(g)), kappa_scat=None,
                                 params=dict(inp.params, n_scat=-1 if w > 0.0 else 0))
        st = iterate_re(i2, max_iter, tol_dT=tol_dT)
        spec = fluxes(i2, T=st["T"], want_spectra=True)[2]
        out = spec * dnu[None, :]
        return dict(T=st["T"], iters=st["iters"], converged=st["converged"], spectrum=spec,
                    reflected=out[:, lam_um < split_um].sum(axis=1), thermal=out[:, lam_um >= split_um].sum(axis=1))

    res = {"absorption": run(0.0, 0.0)}
    for g in g0_values:
        res[float(g)] = run(w0, g)
    return res

