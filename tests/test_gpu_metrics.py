"""Per-column RE metrics and the non-finite guard of the C-ABI (helios_get_re_metrics)."""
import numpy as np
import pytest

from paper_1606_05474_b200 import inputs
from test_gpu_parity import _gpu, _orc

pytestmark = pytest.mark.gpu


def test_per_column_metrics_match_the_oracle():
    b, orc = _gpu(), _orc()
    inp = inputs.make_config(3, n_cols=5, n_bins=30)
    h = b.Helios(inp)
    h.helios_iterate_re(7)
    m = {k: v.cpu().numpy() for k, v in h.helios_get_re_metrics().items()}
    h.close()
    ref = orc.iterate_re(inp, 7)
    pre = orc.iterate_re(inp, 6)                                  # the state the 7th evaluation saw
    Fu, Fd = orc.fluxes(inp, T=pre["T"])
    dF = np.abs(np.diff(Fu - Fd, axis=1))
    sig_T4 = orc.sigma_sb() * pre["T"] ** 4
    dF = np.where(dF < inp.params["flux_floor"] * sig_T4, 0.0, dF)
    assert np.allclose(m["max_dT"], np.max(np.abs(ref["dT_last"]), axis=1), rtol=1e-9, atol=1e-9)
    assert np.allclose(m["max_rel_dF"], np.max(dF / sig_T4, axis=1), rtol=1e-6)
    assert not m["nonfinite"].any()


def test_nonfinite_column_is_flagged_left_alone_and_the_others_carry_on():
    b, orc = _gpu(), _orc()
    inp = inputs.make_config(3, n_cols=4, n_bins=20)
    h = b.Helios(inp)
    T = inp.T0.copy()
    T[2, 10] = np.nan
    h.helios_set_temperatures(T)
    with pytest.raises(b.HeliosError) as e:
        h.helios_iterate_re(3)
    assert e.value.code == b.E_NONFINITE
    m = {k: v.cpu().numpy() for k, v in h.helios_get_re_metrics().items()}
    assert m["nonfinite"].tolist() == [0, 0, 1, 0]
    good = [0, 1, 3]
    ref = orc.iterate_re(inp.take_columns(good), 3)
    # the finite columns advanced exactly as if the bad one were not there (T read through a zero-iteration call,
    # which also shows that the flags are cleared at the start of a call)
    res = h.helios_iterate_re(0)
    assert np.max(np.abs(res["T"].cpu().numpy()[good] - ref["T"])) <= 1e-8
    assert np.isnan(res["T"].cpu().numpy()[2, 10])                   # the flagged column was not touched
    # after the caller repairs the column every call succeeds again
    h.helios_set_temperatures(inp.T0)
    h.helios_fluxes()
    h.helios_iterate_re(2)
    assert not h.helios_get_re_metrics()["nonfinite"].cpu().numpy().any()
    h.close()
