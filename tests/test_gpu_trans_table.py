"""GPU parity of the tabulated transmission function (params.trans_table_dlog10k, S16;
PAPER.md:423) against the oracle's O7b: device and oracle agree on the tabulated path to the usual 1e-10 (fp64) /
1e-4 (fp32), while the tabulated fluxes differ from the exact ones by the approximation's ~1e-3."""
import dataclasses

import numpy as np
import pytest

from paper_1606_05474_b200 import inputs
from test_gpu_parity import ATOL_T, _gpu, _orc, check_fluxes, flux_rel_err, run_fluxes

pytestmark = pytest.mark.gpu


def _tt(inp, dlog=0.1, **kw):
    return dataclasses.replace(inp, params=dict(inp.params, trans_table_dlog10k=dlog, **kw))


def test_trans_table_config1_and_config4_sample_with_spectra():
    check_fluxes(_tt(inputs.make_config(1)), spectra=True)
    check_fluxes(_tt(inputs.make_config(4, n_cols=3)))


@pytest.mark.parametrize("n_layers,n_bins,n_g,n_cols", [(37, 23, 5, 3), (1, 4, 1, 2), (16, 9, 7, 5), (250, 6, 4, 1)])
def test_trans_table_ragged_shapes_direct_and_isothermal_grid(n_layers, n_bins, n_g, n_cols):
    inp = inputs.make_config(4, n_cols=n_cols, n_bins=n_bins, n_layers=n_layers, n_g=n_g)
    w0 = inp.w0.copy()
    w0[0] = 1.0                                                    # an eq. 14 bin among the others
    inp = dataclasses.replace(inp, w0=w0)
    # spectra floor 1e-10 of the column maximum: the BOA value of the eq. 14 bin of a one-layer column is 2e-12 of
    # it, and there the oracle's literal eq. 14 and the algebraically identical (2 F + x F')/(2 + x)
    # differ by 5e-9 of the bin's value on the CPU alone ("Eq. 14 evaluation order")
    check_fluxes(_tt(inp, dlog=0.05), spectra=True, spec_floor=1e-10)
    check_fluxes(_tt(inp, n_scat=-1))
    check_fluxes(_tt(inp, isothermal_layers=1))
    check_fluxes(_tt(inp, planck_table_dT=10.0, planck_table_Tmax=6000.0))      # both tables of PAPER.md:423 together


def test_trans_table_is_an_approximation_of_the_stated_size_and_fp32():
    orc = _orc()
    inp = inputs.make_config(1, n_bins=60)
    ex, tt = run_fluxes(inp), run_fluxes(_tt(inp))
    d = flux_rel_err(tt[0], tt[1], ex[0], ex[1])
    assert 1e-5 < d < 1e-2
    got, ref = run_fluxes(_tt(inp, precision=1)), orc.fluxes(_tt(inp))
    assert flux_rel_err(got[0], got[1], ref[0], ref[1]) <= 1e-4


def test_trans_table_re_steps_and_rejected_combinations():
    b, orc = _gpu(), _orc()
    inp = _tt(inputs.make_config(3, n_cols=3, n_bins=30))
    h = b.Helios(inp)
    out = h.helios_iterate_re(5)
    ref = orc.iterate_re(inp, 5)
    assert np.max(np.abs(out["T"].cpu().numpy() - ref["T"])) <= ATOL_T
    with pytest.raises(b.HeliosError):
        h.helios_set_scattering(np.full(30, 1e-3))
    h.close()
    assert b.helios_workspace_bytes(dict(inp.params, exact_absorption=1)) == 0
    assert b.helios_workspace_bytes(dict(inp.params, trans_table_dlog10k=-0.1)) == 0
