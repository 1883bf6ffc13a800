"""CPU-side checks of the CUDA library (no compute calls): it builds for sm_100a, loads, exports every
symbol include/helios.h declares, validates parameters, and fails loudly without a device."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1606_05474_b200 import binding, build, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "helios.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(helios_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    lib = build.build()
    assert os.path.exists(lib)
    L = ctypes.CDLL(lib)
    syms = declared_symbols()
    assert "helios_setup" in syms and "helios_fluxes" in syms and "helios_iterate_re" in syms
    for s in syms:
        assert hasattr(L, s), f"{s} declared in include/helios.h but not exported"
    assert sorted(binding.EXPORTS) == syms          # the binding mirrors the header one to one


def test_params_struct_matches_header_field_order():
    src = open(os.path.join(ROOT, "include", "helios.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} helios_params;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if decl:
            fields += [f.strip() for f in decl.split(None, 1)[1].split(",")]
    assert fields == [f for f, _ in binding.HeliosParams._fields_]


def test_workspace_bytes_validates_parameters():
    p = inputs.make_config(4).params
    nbytes = binding.helios_workspace_bytes(p)
    # T, step factors, dT, piB, partials, fluxes ... of 8192 columns: a few hundred MB at most
    assert 8192 * 1000 * 8 < nbytes < 2 ** 30
    for bad in (dict(n_layers=0), dict(n_layers=300), dict(warm_start=1), dict(warm_start=2), dict(precision=2), dict(D=0.0),
                dict(ntab_t=1), dict(flux_floor=-1.0), dict(n_scat=-2), dict(n_scat=-1, warm_start=1), dict(exact_absorption=2)):
        assert binding.helios_workspace_bytes(dict(p, **bad)) == 0, bad
    assert binding.helios_workspace_bytes(dict(p, isothermal_layers=1, n_layers=512)) > 0
    assert binding.helios_workspace_bytes(dict(p, n_scat=binding.NSCAT_DIRECT)) == nbytes
    assert binding.helios_workspace_bytes(dict(p, exact_absorption=1)) == nbytes
    # fp32 ray arithmetic keeps an fp32 copy of the k-table in the workspace
    assert binding.helios_workspace_bytes(dict(p, precision=1)) >= 20 * 40 * 1000 * 20 * 4 + 8192 * 1000 * 8   # table copy + pi B(T_intern)


def test_no_device_means_error_not_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(binding.HeliosError) as e:
        binding.Helios(inputs.make_config(0))
    assert e.value.code == binding.E_CUDA
    L = binding.load()
    ctx = ctypes.c_void_p()
    p = binding.params_from_dict(inputs.make_config(0).params)
    dummy = ctypes.c_void_p(256)
    r = L.helios_setup(ctypes.byref(ctx), ctypes.byref(p), *([dummy] * 10), dummy, ctypes.c_size_t(1 << 30), None)
    assert r == binding.E_CUDA and not ctx.value
    assert b"no CUDA device" in L.helios_last_error(None)
    assert binding.helios_measure_fma_peak() == float(binding.E_CUDA)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1606_05474_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("oracle/", "").replace("the oracle", "").replace("test oracle", "") \
                    or f == "inputs.py", f


def test_run_configs_tool_imports_and_fails_loudly_without_a_device(monkeypatch):
    """paper_1606_05474_b200.run_configs (the tool behind profiles/*_configs.md) runs the five BASELINE configs
    through the binding; without a device it raises instead of falling back."""
    import sys
    import torch
    from paper_1606_05474_b200 import run_configs
    assert callable(run_configs.main) and callable(run_configs.run_re) and callable(run_configs.run_flux)
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    monkeypatch.setattr(sys, "argv", ["run_configs", "--configs", "0"])
    with pytest.raises(binding.HeliosError):
        run_configs.main()
