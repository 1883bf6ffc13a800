"""GPU parity of the exact pure-absorption mode (params.exact_absorption, S13):
eq. 4 / eq. 3 with the transmissivity of eq. 6 on the device against the oracle's O8c.
Tolerances as everywhere: interface fluxes <= 1e-10 of the gross flux scale (fp64), <= 1e-4 (fp32)."""
import dataclasses

import numpy as np
import pytest

from paper_1606_05474_b200 import inputs
from test_gpu_parity import ATOL_T, _gpu, _orc, check_fluxes, flux_rel_err, run_fluxes

pytestmark = pytest.mark.gpu


def _exact(inp, **kw):
    return dataclasses.replace(inp, params=dict(inp.params, exact_absorption=1, **kw))


def test_exact_config0_and_config1_shapes_with_spectra():
    check_fluxes(_exact(inputs.make_config(0)), spectra=True)
    check_fluxes(_exact(inputs.make_config(1)), spectra=True)       # w0 > 0 in the inputs: not used in this limit


@pytest.mark.parametrize("n_layers,n_bins,n_g,n_cols", [(37, 23, 5, 3), (1, 4, 1, 2), (16, 9, 7, 5), (250, 6, 4, 1)])
def test_exact_ragged_shapes(n_layers, n_bins, n_g, n_cols):
    check_fluxes(_exact(inputs.make_config(3, n_cols=n_cols, n_bins=n_bins, n_layers=n_layers, n_g=n_g)), spectra=True)


def test_exact_thin_thick_and_isothermal_grid():
    """dtau from ~1e-12 to ~1e9 per sublayer: both branches of E_1, the eq. 3 fallback below dtau_iso,
    transmissivities that underflow; and the isothermal-layer grid (eq. 3 on whole layers)."""
    inp = inputs.make_config(1, n_bins=60)
    for ks in (1e-6, 1e-3, 1.0, 1e3):
        check_fluxes(_exact(dataclasses.replace(inp, kscale=np.array([ks]))))
    check_fluxes(_exact(inputs.make_config(3, n_cols=2, n_bins=40), isothermal_layers=1), spectra=True)


def test_exact_differs_from_two_stream_as_the_paper_says():
    """Section 3.1.5 / Fig. 1: D = 2 is right for thin layers only, so on a column with thick layers the exact
    fluxes differ from the two-stream ones (pure absorption) by more than the parity tolerance, but not wildly."""
    inp = inputs.make_config(0)
    two = run_fluxes(inp)
    ex = run_fluxes(_exact(inp))
    d = flux_rel_err(ex[0], ex[1], two[0], two[1])
    assert 1e-6 < d < 0.3


def test_exact_fp32():
    orc = _orc()
    for inp in (inputs.make_config(0), inputs.make_config(3, n_cols=2, n_bins=50)):
        inp = _exact(inp, precision=1)
        got, ref = run_fluxes(inp), orc.fluxes(inp)
        assert flux_rel_err(got[0], got[1], ref[0], ref[1]) <= 1e-4


def test_exact_re_iterations_match_oracle():
    b, orc = _gpu(), _orc()
    inp = _exact(inputs.make_config(0))
    ref = orc.iterate_re(inp, 10)
    h = b.Helios(inp)
    out = h.helios_iterate_re(10)
    h.synchronize()
    T = out["T"].cpu().numpy()
    h.close()
    assert np.array_equal(out["iters"].cpu().numpy(), ref["iters"])
    assert np.max(np.abs(T - ref["T"])) <= ATOL_T
