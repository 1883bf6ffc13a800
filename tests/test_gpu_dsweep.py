"""GPU parity of the diffusivity-factor experiment of PAPER.md section 3.1.5:
every run of the sweep (exact solver and D = 1.66, 1.8, 1.9, 2) on the device against the oracle's, and the paper's
conclusion from the device's own numbers."""
import numpy as np
import pytest

from paper_1606_05474_b200 import inputs

pytestmark = pytest.mark.gpu


def test_diffusivity_sweep_matches_the_oracle_run_by_run():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test run without a CUDA device (there is no CPU fallback)")
    from paper_1606_05474_b200 import experiments
    from oracle import binding as orc
    inp = inputs.make_config(1, n_bins=40, n_layers=30, n_g=6)
    got = experiments.diffusivity_sweep(inp)
    ref = orc.diffusivity_sweep(inp)
    for k in ref:
        assert np.array_equal(got[k]["converged"], ref[k]["converged"]) and int(ref[k]["converged"][0]) == 1
        assert np.array_equal(got[k]["iters"], ref[k]["iters"]), k
        # free-running RE over a few hundred iterations: 1e-6 K; spectra at the converged profile
        assert np.max(np.abs(got[k]["T"] - ref[k]["T"])) <= 1e-6, k
        s = ref[k]["spectrum"]
        assert np.max(np.abs(got[k]["spectrum"] - s) / np.maximum(s, 1e-12 * s.max())) <= 1e-8, k
    D = (1.66, 1.8, 1.9, 2.0)
    v = [got[d]["spec_mean"] for d in D]
    assert v[0] > v[1] > v[2] > v[3]                           # D = 2 gives the smallest error in the spectrum
    for key in ("dT_rms", "dT_max", "spec_mean", "spec_max"):
        assert all(abs(got[d][key] - ref[d][key]) <= 1e-6 * ref[d][key] for d in D)


def test_scattering_trends_match_the_oracle_run_by_run():
    """PAPER.md:509-517 (Fig. 8): pure absorption and w0 = 0.5 with g0 = -0.5, 0, 0.5, each to radiative equilibrium on
    the device (direct solve) against the oracle's run, and the paper's spectral trends from the device's numbers."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test run without a CUDA device (there is no CPU fallback)")
    from paper_1606_05474_b200 import experiments
    from oracle import binding as orc
    inp = inputs.make_config(1, n_bins=40, n_layers=30, n_g=6)
    got = experiments.scattering_trends(inp)
    ref = orc.scattering_trends(inp)
    for k in ref:
        assert np.array_equal(got[k]["converged"], ref[k]["converged"]) and int(ref[k]["converged"][0]) == 1
        assert np.array_equal(got[k]["iters"], ref[k]["iters"]), k
        assert np.max(np.abs(got[k]["T"] - ref[k]["T"])) <= 1e-6, k           # free-running RE, DESIGN.md section 4
        for q in ("reflected", "thermal"):
            assert abs(got[k][q][0] - ref[k][q][0]) <= 1e-8 * ref[k][q][0], (k, q)
    assert got[-0.5]["reflected"][0] > got[0.0]["reflected"][0] > got[0.5]["reflected"][0] > got["absorption"]["reflected"][0]
    assert got[0.5]["thermal"][0] > got[0.0]["thermal"][0] > got[-0.5]["thermal"][0]
