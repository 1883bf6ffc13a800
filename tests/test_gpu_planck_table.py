"""GPU parity of the tabulated Planck function (params.planck_table_dT, S15;
PAPER.md:423) against the oracle's O4b: the table is an approximation of the exact path, but the device and the
oracle must agree on it to the usual tolerance (<= 1e-10 of the gross flux scale)."""
import dataclasses

import numpy as np
import pytest

from paper_1606_05474_b200 import inputs
from test_gpu_parity import _gpu, _orc, check_fluxes, flux_rel_err, run_fluxes

pytestmark = pytest.mark.gpu


def _tab(inp, dT=10.0, Tmax=6000.0, **kw):
    return dataclasses.replace(inp, params=dict(inp.params, planck_table_dT=dT, planck_table_Tmax=Tmax, **kw))


def test_table_config2_and_config4_sample():
    check_fluxes(_tab(inputs.make_config(2, n_bins=300)), spectra=True)
    check_fluxes(_tab(inputs.make_config(4, n_cols=3, n_bins=200)))


@pytest.mark.parametrize("n_layers,n_bins,n_g,n_cols", [(37, 23, 5, 3), (1, 4, 1, 2), (250, 6, 4, 1)])
def test_table_ragged_shapes_both_grids(n_layers, n_bins, n_g, n_cols):
    inp = inputs.make_config(4, n_cols=n_cols, n_bins=n_bins, n_layers=n_layers, n_g=n_g)
    check_fluxes(_tab(inp, dT=7.5), spectra=True)
    check_fluxes(_tab(inp, dT=25.0, isothermal_layers=1, n_scat=-1))


def test_table_fallback_for_columns_beyond_the_table_and_error_size():
    """Columns with a level at or above planck_table_Tmax use the exact series (bitwise the exact run); the
    others the table; the table run differs from the exact run by the interpolation error (~1e-4 at 10 K)."""
    inp = inputs.make_config(3, n_cols=6, n_bins=40)
    T = inp.T0.copy()
    T[1] *= 3.0                                    # ~2400-6600 K: beyond a 3000 K table
    inp = dataclasses.replace(inp, T0=T)
    ex = run_fluxes(inp)
    tb = run_fluxes(_tab(inp, Tmax=3000.0))
    assert np.array_equal(tb[0][1], ex[0][1]) and np.array_equal(tb[1][1], ex[1][1])
    d = flux_rel_err(np.delete(tb[0], 1, 0), np.delete(tb[1], 1, 0), np.delete(ex[0], 1, 0), np.delete(ex[1], 1, 0))
    assert 1e-8 < d < 1e-3
    check_fluxes(_tab(inp, Tmax=3000.0))


def test_table_fp32_and_re_steps():
    b, orc = _gpu(), _orc()
    inp = _tab(inputs.make_config(1, n_bins=60), precision=1)
    got, ref = run_fluxes(inp), orc.fluxes(inp)
    assert flux_rel_err(got[0], got[1], ref[0], ref[1]) <= 1e-4
    inp = _tab(inputs.make_config(1, n_bins=40))
    h = b.Helios(inp)
    out = h.helios_iterate_re(5)
    h.synchronize()
    T = out["T"].cpu().numpy()
    h.close()
    ref = orc.iterate_re(inp, 5)
    assert np.max(np.abs(T - ref["T"])) <= 1e-8


def test_table_parameters_validated():
    from paper_1606_05474_b200 import binding
    p = inputs.make_config(0).params
    assert binding.helios_workspace_bytes(dict(p, planck_table_dT=10.0, planck_table_Tmax=5.0)) == 0
    assert binding.helios_workspace_bytes(dict(p, planck_table_dT=-1.0)) == 0
    n0 = binding.helios_workspace_bytes(p)
    n1 = binding.helios_workspace_bytes(dict(p, planck_table_dT=10.0, planck_table_Tmax=3000.0))
    assert n1 - n0 >= p["n_bins"] * 302 * 8
