"""RE parity at the samples SURVEY.md section 8(d) prescribes, in the launch plan bench.py times:

  config 4   8192 columns x 1000 bins x 50 iterations on the device, 16 sampled columns against the oracle;
  config 3   1024 columns x 300 bins, 32 sampled columns (100 iterations by default, all iterations to convergence
             with HELIOS_LONG_TESTS=1: ~6 minutes of oracle time);
  lock-step windows of the samples inside a batch large enough for the batch plan (bin chunks, CUDA-graph replay);
  the bare method (flux_floor = 0, no S11 dead zone) in single-step lock-step on configs 0 and 1.
"""
import dataclasses
import os

import numpy as np
import pytest

from paper_1606_05474_b200 import inputs
from test_gpu_parity import ATOL_T, _gpu, _lock_step, _orc, re_sensitivity

pytestmark = pytest.mark.gpu
LONG = os.environ.get("HELIOS_LONG_TESTS", "") == "1"


def _sample(cfg, total, k):
    return np.sort(np.random.default_rng(cfg).choice(total, k, replace=False))


def _batch_free_run(cfg, cols, max_iter, tol_dT, atol_T):
    """The full batch free-running on the device (bench.py's launch shape), the sampled columns on the oracle."""
    b, orc = _gpu(), _orc()
    inp = inputs.make_config(cfg)
    h = b.Helios(inp)
    shape = h.helios_launch_shape()
    out = h.helios_iterate_re(max_iter, tol_dT=tol_dT)
    T, it, cv = (out[k].cpu().numpy() for k in ("T", "iters", "converged"))
    h.close()
    assert np.all(np.isfinite(T))
    ref = orc.iterate_re(inp.take_columns(cols), max_iter, tol_dT=tol_dT)
    assert np.array_equal(cv[cols], ref["converged"])
    d_it = np.abs(it[cols] - ref["iters"])
    if tol_dT > 0.0:
        # free-running to convergence: the stopping test max|dT| < tol_dT is met within a few iterations of the oracle
        # (the trajectories differ by the amounts of DESIGN.md section 4; same allowance as _free_run)
        assert np.all(d_it <= np.maximum(2, ref["iters"] // 50)), (it[cols], ref["iters"])
    else:
        assert not d_it.any()
    per_col = np.max(np.abs(T[cols] - ref["T"]), axis=1)
    same = d_it == 0
    err = float(np.max(per_col[same]))
    print(f"config {cfg}: {len(cols)} sampled columns of {inp.n_cols}, {int(ref['iters'].max())} iterations "
          f"({int((d_it > 0).sum())} columns stop at another iteration than the oracle, by at most {int(d_it.max())}), "
          f"free-run |dT| {err:.2e} K, launch {shape}")
    print("  per-column max |dT| [K], largest first:", np.array2string(np.sort(per_col)[::-1][:8], precision=2),
          " median", f"{np.median(per_col):.2e}")
    # A column that meets the stopping test at another iteration than the oracle's has left the oracle's trajectory
    # (the method's sensitivity: the oracle does the same against itself when its start is moved
    # by 1e-9 K -- test_long_oracle_self_sensitivity_of_config3): few such columns, and a loose bound on them.
    assert (~same).sum() <= max(1, len(cols) // 10) and np.all(per_col[~same] <= 0.5)
    assert err <= atol_T, f"free-run |dT| {err:.3e}"
    return shape, ref


def test_config4_full_batch_50_iterations_16_sampled_columns():
    shape, _ = _batch_free_run(4, _sample(4, 8192, 16), 50, 0.0, atol_T=1e-5)         # measured 1.1e-6 K
    assert shape["grid_x"] == 8192 and shape["grid_y"] == 5 and shape["threads"] == 256


def test_config3_full_batch_32_sampled_columns():
    if LONG:
        # measured: 30 of 32 columns <= 2.9e-6 K (median 8.5e-8 K); two stop 1 and 7 iterations apart, 0.03 / 0.15 K away
        _, ref = _batch_free_run(3, _sample(3, 1024, 32), 20000, 1e-3, atol_T=1e-4)
        assert np.all(ref["converged"] == 1)
    else:
        _batch_free_run(3, _sample(3, 1024, 32), 100, 0.0, atol_T=1e-4)               # measured 5.7e-6 K at 150


def test_config4_lock_step_sample_in_batch_plan():
    """16 sampled columns x 1000 bins tiled to 160 columns: 5 bin chunks, 8 warps, graph replay of the RE loop."""
    inp = inputs.make_config(4).take_columns(_sample(4, 8192, 16))
    worst, allow = _lock_step(inp, 50, 0.0, stride=12, allow_sensitivity=True, tile=10)
    assert worst <= 2e-6 and allow >= worst                                          # measured 4.5e-7 K


def test_config3_lock_step_sample_in_batch_plan():
    inp = inputs.make_config(3).take_columns(_sample(3, 1024, 32)[:16])
    worst, _ = _lock_step(inp, 90, 1e-3, stride=40, allow_sensitivity=True, tile=10)
    assert worst <= 2e-7                                                             # measured 2.2e-8 K


@pytest.mark.parametrize("cfg,stride,windows", [(0, 25, 10), (1, 60, 10)])
def test_bare_method_single_step_lock_step(cfg, stride, windows):
    """The method as printed (flux_floor = 0: no S11 dead zone), one step at a time from the oracle's state.  Eq. 28
    makes the step depend on dF only through sgn(dF)|dF|^0.1, so where dF is rounding noise of the bolometric sums
    (deep, opaque layers: |dF| < 1e-14 of the gross flux) neither side's step is determined; every other layer must
    agree to 1e-8 K plus the first-order sensitivity, and most layers must be of that kind."""
    b, orc = _gpu(), _orc()
    base = inputs.make_config(cfg)
    inp = dataclasses.replace(base, params=dict(base.params, flux_floor=0.0))
    h = b.Helios(inp)
    s = orc.iterate_re(inp, 0)
    worst, compared, total = 0.0, 0, 0
    for _ in range(windows):
        s1 = orc.iterate_re(inp, 1, state=s)
        h.helios_set_temperatures(s["T"])
        h.helios_set_re_state(s["step_factor"], s["sign_hist"], s["iters"], s["converged"])
        T_g = h.helios_iterate_re(1)["T"].cpu().numpy()
        Fu, Fd = orc.fluxes(inp, T=s["T"])
        gross = (np.abs(Fu) + np.abs(Fd))
        dF = np.abs(np.diff(Fu - Fd, axis=1))
        determined = dF > 1e-12 * (gross[:, 1:] + gross[:, :-1])
        err = np.abs(T_g - s1["T"])
        bound = ATOL_T + re_sensitivity(inp, s, Fu, Fd)
        assert np.all(err[determined] <= bound[determined]), f"bare method: |dT| {err[determined].max():.3e}"
        worst = max(worst, float(err[determined].max()))
        compared += int(determined.sum())
        total += determined.size
        s = orc.iterate_re(inp, stride, state=s1)
    h.close()
    print(f"bare method config {cfg}: worst |dT| {worst:.2e} K on {compared} of {total} layer steps")
    assert compared >= 0.6 * total
