"""Runs the five BASELINE.json configurations as they are specified (config 0: 10 RE iterations and RE
to convergence; 1, 3: RE to |dT| < 1e-3 K; 2: one flux evaluation per bin count; 4: 50 RE iterations in
fp64 and fp32) through the C-ABI on cuda:0 and prints iteration counts, wall time and throughput.

    python -m paper_1606_05474_b200.run_configs [--configs 0 1 2 3 4] [--variants [COLS]]

--variants: instead of the configs, the ray kernel's time per RE iteration of config 4 (COLS columns, default 1184) for
every kernel variant and option (sweeps with n_scat = 0 / 1 / 4 / 8, direct solve, albedo per sublayer, Planck and
transmission tables, exact pure-absorption limit; fp64 and fp32), measured with the library's CUDA events.
"""
from __future__ import annotations

import argparse
import dataclasses
import time

import numpy as np

from . import binding, inputs


def run_re(name, inp, max_iter, tol):
    import torch
    warm = binding.Helios(inp)
    warm.helios_iterate_re(2)
    warm.close()
    h = binding.Helios(inp)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    out = h.helios_iterate_re(max_iter, tol_dT=tol)
    h.synchronize()
    dt = time.perf_counter() - t0
    it, cv = out["iters"].cpu().numpy(), out["converged"].cpu().numpy()
    p = inp.params
    upd = float(it.sum()) * p["n_bins"] * p["n_g"] * p["n_layers"]
    print(f"{name}: {p['n_cols']} columns, iterations min/median/max {it.min()}/{int(np.median(it))}/{it.max()}, "
          f"converged {int(cv.sum())}/{len(cv)}, {dt:.3f} s, {it.sum() / dt:.0f} column-iterations/s, "
          f"{upd / dt:.3e} updates/s", flush=True)
    h.close()


def run_flux(name, inp):
    import torch
    h = binding.Helios(inp)
    h.helios_fluxes()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h.synchronize()
    e0.record(h.stream)
    h.helios_fluxes(want_spectra=True)
    e1.record(h.stream)
    h.synchronize()
    ms = e0.elapsed_time(e1)
    p = inp.params
    upd = float(p["n_cols"]) * p["n_bins"] * p["n_g"] * p["n_layers"]
    print(f"{name}: one flux evaluation with spectra, n_scat = {p['n_scat'] if p['n_scat'] >= 0 else 'direct'}: {ms:.3f} ms, {upd / (ms * 1e-3):.3e} updates/s",
          flush=True)
    h.close()


def run_variants(cols):
    base = inputs.make_config(4, n_cols=cols)
    ksc = 30.0 * inputs.rayleigh_h2_kappa(base.bin_edges)
    cases = [("sweeps, n_scat = 0", {"n_scat": 0}, {}), ("sweeps, n_scat = 1", {"n_scat": 1}, {}),
             ("sweeps, n_scat = 4 (config 4 as specified)", {}, {}), ("sweeps, n_scat = 8", {"n_scat": 8}, {}),
             ("direct solve", {"n_scat": binding.NSCAT_DIRECT}, {}),
             ("albedo per sublayer (helios_set_scattering), sweeps", {}, {"kappa_scat": ksc}),
             ("albedo per sublayer, direct solve", {"n_scat": binding.NSCAT_DIRECT}, {"kappa_scat": ksc}),
             ("Planck table, dT = 10 K", {"planck_table_dT": 10.0, "planck_table_Tmax": 6000.0}, {}),
             ("transmission table, dlog10 kappa = 0.1", {"trans_table_dlog10k": 0.1}, {}),
             ("exact pure-absorption limit", {"exact_absorption": 1}, {})]
    p0 = base.params
    upd = float(cols) * p0["n_bins"] * p0["n_g"] * p0["n_layers"]
    for prec, tag in ((0, "fp64"), (1, "fp32")):
        for name, par, kw in cases:
            h = binding.Helios(dataclasses.replace(base, params=dict(p0, precision=prec, **par), **kw))
            for _ in range(2):
                h.helios_iterate_re(1)
            h.helios_enable_timing(True)
            h.helios_kernel_time_ms()
            for _ in range(3):
                h.helios_iterate_re(1)
            ms, n = h.helios_kernel_time_ms()
            h.close()
            print(f"{tag}  {name}: {ms / n:.2f} ms per RE iteration of {cols} columns, {upd / (ms / n * 1e-3):.3e} updates/s", flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="*", default=[0, 1, 2, 3, 4])
    ap.add_argument("--variants", type=int, nargs="?", const=1184, default=None)
    args = ap.parse_args()
    if args.variants:
        run_variants(args.variants)
        return
    if 0 in args.configs:
        run_flux("config 0", inputs.make_config(0))
        run_re("config 0 (RE to |dT| < 1e-3 K)", inputs.make_config(0), 5000, 1e-3)
    if 1 in args.configs:
        run_re("config 1 (RE to |dT| < 1e-3 K)", inputs.make_config(1), 20000, 1e-3)
        c1 = inputs.make_config(1)
        run_re("config 1, direct solve (RE to |dT| < 1e-3 K)",
               dataclasses.replace(c1, params=dict(c1.params, n_scat=binding.NSCAT_DIRECT)), 20000, 1e-3)
    if 2 in args.configs:
        for nb in (300, 1000, 3000):
            run_flux(f"config 2, {nb} bins", inputs.make_config(2, n_bins=nb))
        # the same evaluations with the direct coupled solve in place of the 1 + 80 sweeps (S12)
        for nb in (300, 1000, 3000):
            i2 = inputs.make_config(2, n_bins=nb)
            run_flux(f"config 2, {nb} bins, direct solve",
                     dataclasses.replace(i2, params=dict(i2.params, n_scat=binding.NSCAT_DIRECT)))
    if 3 in args.configs:
        run_re("config 3 (RE to |dT| < 1e-3 K)", inputs.make_config(3), 20000, 1e-3)
    if 4 in args.configs:
        c4 = inputs.make_config(4)
        run_re("config 4 fp64 (50 RE iterations)", c4, 50, 0.0)
        run_re("config 4 fp32 (50 RE iterations)", dataclasses.replace(c4, params=dict(c4.params, precision=1)), 50, 0.0)
        run_re("config 4 fp64, direct solve (50 RE iterations)",
               dataclasses.replace(c4, params=dict(c4.params, n_scat=binding.NSCAT_DIRECT)), 50, 0.0)


if __name__ == "__main__":
    main()
