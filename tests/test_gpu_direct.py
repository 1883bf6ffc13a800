"""GPU parity of the direct coupled solve (n_scat = HELIOS_NSCAT_DIRECT, S12):
the CUDA path (adding method scanned over the lanes of a warp) against the oracle's O8b (Gaussian
elimination of the same system), element by element on the same seeded inputs.  Tolerances as for the
sweeps: interface fluxes <= 1e-10 relative to the gross flux scale of the interface (fp64), <= 1e-4 (fp32)."""
import dataclasses

import numpy as np
import pytest

from paper_1606_05474_b200 import inputs
from test_gpu_parity import RTOL_FLUX, ATOL_T, _gpu, _orc, check_fluxes, flux_rel_err, run_fluxes

pytestmark = pytest.mark.gpu

RTOL_FLUX_F32 = 1e-4
DIRECT = -1


def _direct(inp, **kw):
    return dataclasses.replace(inp, params=dict(inp.params, n_scat=DIRECT, **kw))


def test_direct_config1_full_size_with_spectra():
    check_fluxes(_direct(inputs.make_config(1)), spectra=True)


def test_direct_config4_physics_sample():
    check_fluxes(_direct(inputs.make_config(4, n_cols=3)))


@pytest.mark.parametrize("n_layers,n_bins,n_g,n_cols", [(37, 23, 5, 3), (1, 4, 1, 2), (16, 9, 7, 5),
                                                        (3, 2, 3, 1), (64, 12, 20, 2), (250, 6, 4, 1)])
def test_direct_ragged_shapes(n_layers, n_bins, n_g, n_cols):
    check_fluxes(_direct(inputs.make_config(4, n_cols=n_cols, n_bins=n_bins, n_layers=n_layers, n_g=n_g)),
                 spectra=True)


def test_direct_isothermal_layers_and_pure_scattering_bins():
    iso = inputs.make_config(4, n_cols=2, n_bins=40, n_layers=100)
    check_fluxes(_direct(iso, isothermal_layers=1), spectra=True)
    ps = inputs.make_config(4, n_cols=2, n_bins=12, n_layers=30)
    w0 = ps.w0.copy()
    w0[::3] = 1.0
    w0[1] = 1.0 - 1e-7
    check_fluxes(_direct(dataclasses.replace(ps, w0=w0)), spectra=True)


def test_direct_thin_and_thick_columns():
    inp = inputs.make_config(1, n_bins=60)
    for ks in (1e-6, 1e-3, 1e3):
        check_fluxes(_direct(dataclasses.replace(inp, kscale=np.array([ks]))))


def test_direct_pure_absorption_equals_one_sweep_bitwise():
    """Every w0 == 0: the coupled system is triangular, one sweep is exact and the direct flag changes nothing."""
    inp = inputs.make_config(0)
    a = run_fluxes(inp)
    b = run_fluxes(_direct(inp))
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_direct_is_the_limit_of_the_gpu_sweeps():
    """The GPU's own sweeps converge to the GPU's direct solve: config 2 physics, 80 extra sweeps
    leave <= 1e-6 (the paper's one-shot setting), 400 leave <= 1e-12."""
    inp = inputs.make_config(2, n_bins=300)
    d = run_fluxes(_direct(inp))
    s80 = run_fluxes(inp)
    s400 = run_fluxes(dataclasses.replace(inp, params=dict(inp.params, n_scat=400)))
    assert flux_rel_err(s80[0], s80[1], d[0], d[1]) <= 1e-6
    assert flux_rel_err(s400[0], s400[1], d[0], d[1]) <= 1e-12


def test_direct_near_conservative_scattering():
    """w0 up to 1 - 2e-6 (just below the eq. 14 switch): 1 - rt rb of the adding method loses digits like the
    system's own conditioning does; the oracle's elimination and the GPU still agree to 1e-10."""
    rng = np.random.default_rng(77)
    inp = inputs.make_config(4, n_cols=2, n_bins=16, n_layers=60)
    w0 = 1.0 - 10.0 ** rng.uniform(-5.7, -1, 16)
    check_fluxes(_direct(dataclasses.replace(inp, w0=w0, g0=rng.uniform(-0.5, 0.9, 16))))


def test_direct_fp32():
    b, orc = _gpu(), _orc()
    for inp in (inputs.make_config(1), inputs.make_config(4, n_cols=3, n_bins=100),
                inputs.make_config(4, n_cols=2, n_bins=9, n_layers=37, n_g=5)):
        inp = _direct(inp, precision=1)
        got = run_fluxes(inp)
        ref = orc.fluxes(inp)
        assert np.all(np.isfinite(got[0])) and np.all(np.isfinite(got[1]))
        assert flux_rel_err(got[0], got[1], ref[0], ref[1]) <= RTOL_FLUX_F32


def test_direct_randomised_sweep():
    b, orc = _gpu(), _orc()
    rng = np.random.default_rng(20260511)
    worst = 0.0
    for case in range(60):
        cfg = int(rng.choice([1, 3, 4]))
        n = int(rng.choice([1, 2, 3, 5, 8, 16, 17, 31, 32, 33, 48, 64, 100, 101, 128, 200, 256]))
        iso = int(rng.random() < 0.25)
        nb, ng, nc = int(rng.integers(1, 30)), int(rng.choice([1, 2, 3, 4, 5, 8, 20])), int(rng.integers(1, 4))
        inp = inputs.make_config(cfg, n_cols=nc, n_bins=nb, n_layers=n, n_g=ng)
        w0, g0 = inp.w0.copy(), inp.g0.copy()
        mode = int(rng.integers(0, 3))
        if mode == 1:
            w0, g0 = rng.uniform(0, 1, nb), rng.uniform(-0.9, 0.9, nb)
        if mode == 2:
            w0 = np.where(rng.random(nb) < 0.3, 1.0, rng.uniform(0.9, 0.9999, nb))
            g0 = rng.uniform(-0.5, 0.9, nb)
        if not np.any(w0 > 0):
            w0[0] = 0.5
        inp = dataclasses.replace(inp, w0=w0, g0=g0, kscale=inp.kscale * 10.0 ** rng.uniform(-5, 3, nc),
                                  t_intern=np.where(rng.random(nc) < 0.5, 0.0, rng.uniform(50, 900, nc)))
        inp = _direct(inp, isothermal_layers=iso, D=float(rng.choice([2.0, 1.66])))
        ref = orc.fluxes(inp)
        got = run_fluxes(inp)
        sc = np.maximum(np.abs(ref[0]), np.abs(ref[1]))
        sc = np.maximum(sc, 1e-12 * np.max(sc, axis=1, keepdims=True) + 1e-300)
        e = max(np.max(np.abs(got[0] - ref[0]) / sc), np.max(np.abs(got[1] - ref[1]) / sc))
        worst = max(worst, e)
        assert e <= RTOL_FLUX, f"case {case}: rel err {e:.3e} (n={n}, iso={iso}, mode={mode}, nb={nb}, ng={ng})"
    print("direct randomised sweep: worst rel err", worst)


def test_direct_re_iterations_match_oracle():
    b, orc = _gpu(), _orc()
    inp = _direct(inputs.make_config(1, n_bins=60))
    ref = orc.iterate_re(inp, 5)
    h = b.Helios(inp)
    out = h.helios_iterate_re(5)
    h.synchronize()
    T = out["T"].cpu().numpy()
    h.close()
    assert np.array_equal(out["iters"].cpu().numpy(), ref["iters"])
    assert np.max(np.abs(T - ref["T"])) <= ATOL_T


def test_direct_rejects_warm_start():
    b = _gpu()
    inp = _direct(inputs.make_config(1, n_bins=8), warm_start=1)
    with pytest.raises(b.HeliosError) as e:
        b.Helios(inp)
    assert e.value.code == b.E_BADARG


def test_direct_config4_full_size_sampled_columns():
    """BASELINE configs[4] at full size in bench.py's launch shape with the direct solve; sampled columns
    against the oracle, plus the properties that hold at any size."""
    b, orc = _gpu(), _orc()
    inp = _direct(inputs.make_config(4))
    sample = [0, 8191, 4242]
    h = b.Helios(inp)
    shape = h.helios_launch_shape()
    Fu, Fd = h.helios_fluxes()
    h.synchronize()
    Fu, Fd = Fu.cpu().numpy(), Fd.cpu().numpy()
    h.close()
    assert shape["grid_x"] == 8192 and shape["grid_y"] == 5 and shape["S"] == 13 and shape["threads"] == 256
    assert np.all(np.isfinite(Fu)) and np.all(np.isfinite(Fd))
    Ru, Rd = orc.fluxes(inp.take_columns(sample))
    assert flux_rel_err(Fu[sample], Fd[sample], Ru, Rd) <= RTOL_FLUX
    top = np.sum(np.diff(inp.bin_edges) * inp.f_star) * inp.f_star_scale
    assert np.allclose(Fd[:, -1], top, rtol=1e-12)
    assert np.all(Fu >= 0) and np.all(Fd >= 0)
    # eq. 22 summed over bins and g: F_up(BOA) - F_dn(BOA) = pi B(T_intern) >= 0
    assert np.all(Fu[:, 0] - Fd[:, 0] >= -1e-12 * np.abs(Fd[:, 0]))


def test_direct_config1_re_lock_step():
    """Lock-step RE parity with the direct solve in every evaluation."""
    from test_gpu_parity import _lock_step
    inp = _direct(inputs.make_config(1, n_bins=30))
    assert _lock_step(inp, 200, 1e-3)[0] <= 1e-8
