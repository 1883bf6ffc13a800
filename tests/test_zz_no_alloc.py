"""helios_fluxes_static: the flux evaluation for callers that must not allocate (include/helios.h).  The ray
kernel's partial sums go to the library's file-scope static device array instead of the workspace; the output
must equal helios_fluxes' on two calls in a row (the array keeps the previous call's contents), sizes beyond
HELIOS_STATIC_SCRATCH_BYTES must be rejected, and the call must not allocate device memory.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other
tests."""
import numpy as np
import pytest

from paper_1606_05474_b200 import inputs
from test_gpu_parity import RTOL_FLUX, _gpu, _orc, flux_rel_err

pytestmark = pytest.mark.gpu

STATIC_SCRATCH_BYTES = 4 * 1024 * 1024      # HELIOS_STATIC_SCRATCH_BYTES of include/helios.h


def _cases():
    return [inputs.make_config(0),                                                   # one column, pure absorption
            inputs.make_config(1, n_bins=75),                                        # one column, bins over many blocks, unit-split plan
            inputs.make_config(4, n_cols=5, n_bins=24, n_layers=37, n_g=6)]          # ragged scattering batch


@pytest.mark.parametrize("case", range(3))
def test_static_scratch_entry_point_equals_the_workspace_path_on_two_calls_in_a_row(case):
    import torch
    b = _gpu()
    inp = _cases()[case]
    h = b.Helios(inp)
    shape = h.helios_launch_shape()
    assert shape["grid_y"] * h.nc * 4 * (h.n + 1) * 8 <= STATIC_SCRATCH_BYTES
    T1 = inp.T0
    T2 = inp.T0 * np.linspace(0.9, 1.15, h.n)[None, :]           # second call: other temperatures, stale scratch
    out = (h.empty(h.nc, h.n + 1), h.empty(h.nc, h.n + 1))       # the caller's buffers, allocated before the calls
    ref, got = [], []
    for T in (T1, T2):
        h.helios_set_temperatures(T)
        ref.append([x.cpu().numpy() for x in h.helios_fluxes()])
    h.synchronize()
    h.helios_set_temperatures(T1)
    before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    h.helios_fluxes_static(out)                                   # two calls in a row, no synchronisation between
    h.helios_fluxes_static(out)
    h.synchronize()
    assert torch.cuda.memory_allocated() == before[0]                                   # nothing went through torch ...
    assert before[1] - torch.cuda.mem_get_info()[0] < (1 << 20)                         # ... nor past it (cudaMalloc granule: 2 MiB)
    got.append([x.cpu().numpy() for x in out])
    h.helios_set_temperatures(T2)
    h.helios_fluxes_static(out)
    h.synchronize()
    got.append([x.cpu().numpy() for x in out])
    # the workspace path was not disturbed by the static one
    again = [x.cpu().numpy() for x in h.helios_fluxes()]
    h.close()
    for (Fu, Fd), (Ru, Rd) in zip(got, ref):
        assert np.all(np.isfinite(Fu)) and np.all(np.isfinite(Fd))
        assert flux_rel_err(Fu, Fd, Ru, Rd) <= RTOL_FLUX
        assert np.array_equal(Fu, Ru) and np.array_equal(Fd, Rd)   # same kernels, same summation order
    assert np.array_equal(again[0], ref[1][0]) and np.array_equal(again[1], ref[1][1])
    # ... and both agree with the oracle (the bar of the parity tests)
    Ou, Od = _orc().fluxes(inp, T=T2)
    assert flux_rel_err(got[1][0], got[1][1], Ou, Od) <= RTOL_FLUX


def test_static_scratch_entry_point_rejects_shapes_beyond_its_maximum():
    b = _gpu()
    inp = inputs.make_config(3, n_cols=1400, n_bins=16, n_g=4)    # 1400 x 4 x 101 x 8 B = 4.5 MB of partial sums
    h = b.Helios(inp)
    shape = h.helios_launch_shape()
    assert shape["grid_y"] * h.nc * 4 * (h.n + 1) * 8 > STATIC_SCRATCH_BYTES
    out = (h.empty(h.nc, h.n + 1), h.empty(h.nc, h.n + 1))
    with pytest.raises(b.HeliosError) as e:
        h.helios_fluxes_static(out)
    assert e.value.code == b.E_WORKSPACE
    assert "HELIOS_STATIC_SCRATCH_BYTES" in str(e.value) and str(STATIC_SCRATCH_BYTES) in str(e.value)
    Fu, Fd = h.helios_fluxes()                                    # the context is still usable
    h.synchronize()
    assert np.all(np.isfinite(Fu.cpu().numpy())) and np.all(np.isfinite(Fd.cpu().numpy()))
    h.close()
