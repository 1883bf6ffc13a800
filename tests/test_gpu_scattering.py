"""GPU parity of the single-scattering albedo per sublayer (helios_set_scattering, SURVEY.md 8(f)4,
DESIGN.md S14) against the oracle: interface fluxes <= 1e-10 of the gross flux scale
(fp64), <= 1e-4 (fp32); RE temperatures <= 1e-8 K over a few iterations."""
import dataclasses

import numpy as np
import pytest

from paper_1606_05474_b200 import inputs
from test_gpu_parity import ATOL_T, _gpu, _orc, check_fluxes, flux_rel_err, run_fluxes

pytestmark = pytest.mark.gpu


def _rayleigh(inp, boost=1.0, **kw):
    return dataclasses.replace(inp, kappa_scat=boost * inputs.rayleigh_h2_kappa(inp.bin_edges),
                               params=dict(inp.params, **kw))


def test_rayleigh_config1_full_size_with_spectra():
    check_fluxes(_rayleigh(inputs.make_config(1)), spectra=True)


def test_rayleigh_direct_and_sweeps_agree_with_their_oracles():
    inp = _rayleigh(inputs.make_config(1, n_bins=80), boost=30.0)
    check_fluxes(inp)
    check_fluxes(dataclasses.replace(inp, params=dict(inp.params, n_scat=-1)), spectra=True)


@pytest.mark.parametrize("n_layers,n_bins,n_g,n_cols", [(37, 23, 5, 3), (1, 4, 1, 2), (16, 9, 7, 5), (250, 6, 4, 1)])
def test_scattering_ragged_shapes_with_g0(n_layers, n_bins, n_g, n_cols):
    """config 4 physics (g0 != 0 per bin) with a random scattering opacity spanning w0 from ~0 to ~1, including
    bins whose sublayers fall on the eq. 14 side of the switch."""
    inp = inputs.make_config(4, n_cols=n_cols, n_bins=n_bins, n_layers=n_layers, n_g=n_g)
    rng = np.random.default_rng(n_layers)
    ks = 10.0 ** rng.uniform(-8, 3, n_bins)
    ks[0] = 1e12                                   # 1 - w0 < 1e-6 everywhere in this bin
    check_fluxes(dataclasses.replace(inp, kappa_scat=ks), spectra=True)
    check_fluxes(dataclasses.replace(inp, kappa_scat=ks, params=dict(inp.params, n_scat=-1)))


def test_scattering_isothermal_grid_and_zero_opacity():
    inp = inputs.make_config(4, n_cols=2, n_bins=30)
    check_fluxes(_rayleigh(inp, boost=100.0, isothermal_layers=1), spectra=True)
    z = dataclasses.replace(inp, kappa_scat=np.zeros(30))
    check_fluxes(z)
    a = run_fluxes(z)
    b = run_fluxes(dataclasses.replace(inp, w0=np.zeros(30)))
    assert flux_rel_err(a[0], a[1], b[0], b[1]) <= 1e-13           # all zeros = pure absorption


def test_scattering_fp32():
    orc = _orc()
    inp = _rayleigh(inputs.make_config(1, n_bins=100), boost=10.0, precision=1)
    got, ref = run_fluxes(inp), orc.fluxes(inp)
    assert flux_rel_err(got[0], got[1], ref[0], ref[1]) <= 1e-4


def test_scattering_re_iterations_and_graph_invalidation():
    """RE steps with the scattering opacity set AFTER a first graph-replayed RE call on the same context."""
    b, orc = _gpu(), _orc()
    base = inputs.make_config(1, n_bins=40)
    inp = _rayleigh(base, boost=20.0)
    h = b.Helios(base)
    h.helios_iterate_re(32)                        # captures the CUDA graph without scattering opacity
    h.helios_set_scattering(inp.kappa_scat)
    h.helios_set_columns(inp.T0, inp.f_star, inp.f_star_scale, inp.t_intern, inp.kscale)   # restart
    out = h.helios_iterate_re(20)
    h.synchronize()
    T = out["T"].cpu().numpy()
    h.close()
    ref = orc.iterate_re(inp, 20)
    assert np.array_equal(out["iters"].cpu().numpy(), ref["iters"])
    assert np.max(np.abs(T - ref["T"])) <= 1e-6    # 20 free-running steps


def test_scattering_rejected_in_exact_limit():
    b = _gpu()
    inp = inputs.make_config(0)
    inp = dataclasses.replace(inp, params=dict(inp.params, exact_absorption=1), kappa_scat=np.ones(16))
    with pytest.raises(b.HeliosError) as e:
        b.Helios(inp)
    assert e.value.code == b.E_BADARG
