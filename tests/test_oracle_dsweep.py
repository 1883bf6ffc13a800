"""The diffusivity-factor experiment of PAPER.md section 3.1.5 (Fig. 11) with the oracle: two-stream
radiative-equilibrium profiles for D = 1.66, 1.8, 1.9, 2 against the exact pure-absorption solution (eq. 3-6).  Pins
the paper's conclusion and thereby the D-dependence of the two-stream path (eq. 8, 2 pi eps B sources) against the
D-free exact path.  CPU only."""
import dataclasses

import numpy as np

from oracle import binding as orc
from paper_1606_05474_b200 import inputs


def column():
    """config-1-like column (stellar heating, 1e-6 ... 1e3 bar), shrunk so that five RE runs take seconds."""
    return inputs.make_config(1, n_bins=40, n_layers=30, n_g=6)


def test_D2_is_closest_to_the_exact_solution_and_the_error_falls_monotonically_with_D():
    res = orc.diffusivity_sweep(column())
    assert all(int(res[k]["converged"][0]) == 1 for k in res)
    D = (1.66, 1.8, 1.9, 2.0)
    rms = [res[d]["dT_rms"] for d in D]
    spec = [res[d]["spec_mean"] for d in D]
    # PAPER.md:551 (the GJ 1214b case of Fig. 11): "Regarding temperature, the D = 1.9 and 2 models produce the best
    # match to the exact solution.  However, D = 2 leads, on average, to the smallest error in the spectrum";
    # Amundsen et al.'s 1.66 is the worst of the four
    assert rms[0] > rms[1] > max(rms[2], rms[3])
    assert abs(rms[2] - rms[3]) < 0.15 * rms[3] and rms[3] < 0.3 * rms[0]
    assert spec[0] > spec[1] > spec[2] > spec[3]
    assert spec[3] < 0.25 * spec[2] and spec[3] < 0.06 * spec[0] and res[2.0]["spec_max"] < 0.05
    # "we expect the diffusivity factor to approach a value of 2 when the vertical resolution of the model is
    # sufficient": doubling the layer count brings the D = 2 spectrum closer to the exact one
    fine = orc.diffusivity_sweep(inputs.make_config(1, n_bins=40, n_layers=60, n_g=6), D_values=(2.0,))
    assert fine[2.0]["spec_mean"] < 0.85 * res[2.0]["spec_mean"]


def test_sweep_ignores_scattering_inputs_and_D_does_not_enter_the_exact_run():
    """The experiment is defined in the pure-absorption limit: w0 of the inputs is dropped, and the exact solver has no
    D ("there is no need to specify D")."""
    inp = column()
    a = orc.diffusivity_sweep(inp, D_values=(2.0,), max_iter=5, tol_dT=0.0)
    b = orc.diffusivity_sweep(dataclasses.replace(inp, w0=np.zeros(40), params=dict(inp.params, D=1.7)), D_values=(2.0,),
                              max_iter=5, tol_dT=0.0)
    assert np.array_equal(a["exact"]["T"], b["exact"]["T"]) and np.array_equal(a[2.0]["T"], b[2.0]["T"])
