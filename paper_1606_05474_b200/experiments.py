"""Two consistency experiments of the paper on the CUDA path: the diffusivity-factor experiment of section 3.1.5
(Fig. 11) and the scattering trends of section 3.1.2 (Fig. 8).

"One may obtain an exact solution of the radiative transfer equation, without invoking the two-stream
approximation, only in the limit of pure absorption.  This solution may be compared to two-stream calculations with
different assumed values of the diffusivity factor": a purely absorbing column is iterated to radiative equilibrium
with the two-stream solver for D = 1.66, 1.8, 1.9 and 2 and with the exact solver (params.exact_absorption, eq. 3-6),
and temperature profiles and emission spectra are compared with the exact run.

Only calls of the C-ABI binding and statistics of what they return; no arithmetic of the method lives here.
"""
from __future__ import annotations

import dataclasses

import numpy as np

from . import binding

PAPER_D_VALUES = (1.66, 1.8, 1.9, 2.0)


def _pure_absorption(inp, **params):
    nb = inp.params["n_bins"]
    return dataclasses.replace(inp, w0=np.zeros(nb), g0=np.zeros(nb), kappa_scat=None,
                               params=dict(inp.params, n_scat=0, **params))


def _run(inp, max_iter, tol_dT, device):
    h = binding.Helios(inp, device=device)
    try:
        out = h.helios_iterate_re(max_iter, tol_dT=tol_dT)
        T = out["T"].cpu().numpy()
        h.helios_set_temperatures(T)
        _, _, spec_up, _ = h.helios_fluxes(want_spectra=True)
        h.synchronize()
        return dict(T=T, iters=out["iters"].cpu().numpy(), converged=out["converged"].cpu().numpy(),
                    spectrum=spec_up.cpu().numpy())
    finally:
        h.close()


def diffusivity_sweep(inp, D_values=PAPER_D_VALUES, max_iter=20000, tol_dT=1.0e-3, device="cuda:0"):
    """Returns {"exact": run, D: run, ...}; every two-stream run carries its deviation from the exact one:
    max and rms temperature difference [K] and the mean / max relative difference of the TOA emission spectrum
    (bins below 1e-3 of the brightest one are judged against that floor)."""
    res = {"exact": _run(_pure_absorption(inp, exact_absorption=1), max_iter, tol_dT, device)}
    ex = res["exact"]
    floor = 1.0e-3 * np.max(ex["spectrum"], axis=1, keepdims=True)
    for D in D_values:
        r = _run(_pure_absorption(inp, exact_absorption=0, D=float(D)), max_iter, tol_dT, device)
        dT = r["T"] - ex["T"]
        ds = np.abs(r["spectrum"] - ex["spectrum"]) / np.maximum(ex["spectrum"], floor)
        r.update(dT_max=float(np.max(np.abs(dT))), dT_rms=float(np.sqrt(np.mean(dT * dT))),
                 spec_mean=float(np.mean(ds)), spec_max=float(np.max(ds)))
        res[float(D)] = r
    return res


PAPER_G0_VALUES = (-0.5, 0.0, 0.5)


def scattering_trends(inp, w0=0.5, g0_values=PAPER_G0_VALUES, split_um=1.0, max_iter=20000, tol_dT=1.0e-3,
                      device="cuda:0"):
    """"we set w0 = 0.5 across all wavelengths.  We then examine models with g0 = -0.5, 0 and 0.5"
    against "the fiducial pure absorption model".  Every model is iterated to radiative equilibrium (coupled system
    solved, HELIOS_NSCAT_DIRECT); returns {"absorption": run, g0: run}, each with T, iters, converged, the TOA emission
    spectrum at the converged profile and its integrals below / above split_um ("reflected light at <~ 1 um", "thermal
    emission at >~ 1 um")."""
    nb = inp.params["n_bins"]
    lam_um = 1.0e4 / (0.5 * (inp.bin_edges[:-1] + inp.bin_edges[1:]))
    dnu = np.diff(inp.bin_edges)
    res = {}
    for key, w, g in [("absorption", 0.0, 0.0)] + [(float(g), w0, g) for g in g0_values]:
        i2 = dataclasses.replace(inp, w0=np.full(nb, float(w)), g0=np.full(nb, float(g)), kappa_scat=None,
                                 params=dict(inp.params, n_scat=binding.NSCAT_DIRECT if w > 0.0 else 0))
        r = _run(i2, max_iter, tol_dT, device)
        out = r["spectrum"] * dnu[None, :]
        r.update(reflected=out[:, lam_um < split_um].sum(axis=1), thermal=out[:, lam_um >= split_um].sum(axis=1))
        res[key] = r
    return res

