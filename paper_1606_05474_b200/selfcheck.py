"""Self-check of the CUDA path: one small launch of every kernel variant and launch plan.

  python -m paper_1606_05474_b200.selfcheck [--list] [case ...]

Runs each case through the C-ABI on cuda:0 and checks what holds without a reference: every output is
finite, fluxes are non-negative, F_dn at the top equals the stellar input (eq. 20), a
repeated call gives bitwise the same result, RE counters advance.  It compares with no reference (the parity
tests under tests/ do that); its purpose is to put every code path of the library under a tool such as

  compute-sanitizer --tool memcheck  python -m paper_1606_05474_b200.selfcheck
  compute-sanitizer --tool racecheck python -m paper_1606_05474_b200.selfcheck

(the ray kernel re-uses shared-memory regions under __syncwarp ordering: the kappa stage doubles as the
Planck stage, the spectrum buffer sits behind the per-warp regions), or under the library's own checked build
(`python -m paper_1606_05474_b200.build --checked`: NaN-poisoned shared memory, guard words, index checks).  Each
case prints a digest of its outputs: a checked and an ordinary build must print the same ones.
Exit code 0 = all cases passed.
"""
from __future__ import annotations

import dataclasses
import hashlib
import sys

import numpy as np

from . import binding, inputs


def _cases():
    mk = inputs.make_config
    rep = dataclasses.replace

    def par(inp, **kw):
        return rep(inp, params=dict(inp.params, **kw))

    ragged = mk(4, n_cols=3, n_bins=24, n_layers=37, n_g=6)
    c = {}
    c["config0"] = (mk(0), dict(spectra=True, re=10))                      # one block, pure absorption
    c["config1_gsplit"] = (mk(1, n_bins=60), dict(spectra=True, re=20))       # bins shared by warps (unit-split plan), graph replay
    c["ragged_cfg4"] = (ragged, dict(spectra=True, re=5))                     # ragged tails everywhere, g0 != 0
    c["ragged_cfg4_fp32"] = (par(ragged, precision=1), dict(spectra=True, re=5))
    c["direct"] = (par(ragged, n_scat=binding.NSCAT_DIRECT), dict(spectra=True, re=3))
    c["direct_fp32"] = (par(ragged, n_scat=binding.NSCAT_DIRECT, precision=1), dict(spectra=True))
    c["iso_layers"] = (par(mk(4, n_cols=2, n_bins=40, n_layers=100), isothermal_layers=1, n_scat=12), dict(spectra=True))
    c["tall_S13"] = (mk(4, n_cols=1, n_bins=6, n_layers=200, n_g=4), dict(spectra=True, re=2))
    c["tall_S16_fp32"] = (par(mk(4, n_cols=1, n_bins=6, n_layers=250, n_g=4), precision=1), dict())
    ps = mk(4, n_cols=2, n_bins=12, n_layers=30)
    w0 = ps.w0.copy()
    w0[::3] = 1.0
    c["pure_scattering_eq14"] = (rep(par(ps, n_scat=30), w0=w0), dict(spectra=True))
    c["exact_absorption"] = (par(ragged, exact_absorption=1), dict(spectra=True, re=3))          # alt variant
    sc = rep(ragged, kappa_scat=30.0 * inputs.rayleigh_h2_kappa(ragged.bin_edges))
    c["scattering_opacity"] = (sc, dict(spectra=True, re=3))                                      # alt variant
    c["scattering_opacity_direct_fp32"] = (par(sc, n_scat=binding.NSCAT_DIRECT, precision=1), dict())
    c["planck_table"] = (par(ragged, planck_table_dT=10.0, planck_table_Tmax=4000.0), dict(spectra=True, re=3))   # tab variant
    c["planck_table_fp32"] = (par(ragged, planck_table_dT=10.0, planck_table_Tmax=4000.0, precision=1), dict())
    c["warm_start"] = (par(mk(1, n_bins=20), warm_start=1, n_scat=2), dict(re=6))
    c["batch_chunks"] = (mk(4, n_cols=150, n_bins=200, n_layers=20, n_g=4), dict(re=2))           # batch plan: several bin chunks
    return c


def run_case(name, inp, spectra=False, re=0):
    h = binding.Helios(inp, device="cuda:0")
    try:
        out = [o.cpu().numpy() for o in h.helios_fluxes(want_spectra=spectra)]
        again = [o.cpu().numpy() for o in h.helios_fluxes(want_spectra=spectra)]
        for a, b in zip(out, again):
            if not np.array_equal(a, b):
                raise RuntimeError(f"{name}: repeated evaluation differs")
        for a in out:
            if not np.all(np.isfinite(a)):
                raise RuntimeError(f"{name}: non-finite output")
        tol = 1e-5 if inp.params["precision"] else 1e-12
        if not (np.all(out[0] >= 0) and np.all(out[1] >= 0)):
            raise RuntimeError(f"{name}: negative flux")
        top = np.sum(np.diff(inp.bin_edges) * inp.f_star) * inp.f_star_scale
        if not np.allclose(out[1][:, -1], top, rtol=tol, atol=1e-300):
            raise RuntimeError(f"{name}: F_dn(TOA) is not the stellar input")
        if re:
            r = h.helios_iterate_re(re)
            st = h.helios_get_re_state()
            T = r["T"].cpu().numpy()
            if not np.all(np.isfinite(T)) or not np.all(r["iters"].cpu().numpy() == re):
                raise RuntimeError(f"{name}: RE iteration failed")
            if not np.all(np.isfinite(st["step_factor"].cpu().numpy())):
                raise RuntimeError(f"{name}: RE state non-finite")
        digest = hashlib.sha1(b"".join(np.ascontiguousarray(a).tobytes() for a in out)).hexdigest()[:12]
        shape = h.helios_launch_shape()
        print(f"selfcheck {name}: ok  sha1={digest}  grid=({shape['grid_x']},{shape['grid_y']}) threads={shape['threads']} "
              f"smem={shape['smem']} S={shape['S']} launches={h.helios_launch_count()}", flush=True)
    finally:
        h.close()


def main(argv):
    cases = _cases()
    if "--list" in argv:
        print("\n".join(cases))
        return 0
    names = [a for a in argv if not a.startswith("-")] or list(cases)
    for n in names:
        inp, kw = cases[n]
        run_case(n, inp, **kw)
    print(f"selfcheck: {len(names)} cases passed")
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1:]))
