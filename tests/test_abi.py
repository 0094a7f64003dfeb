"""The C-ABI library builds, loads and exports every symbol include/vpmc.h declares (no compute calls: no GPU here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "vpmc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vpmc_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    syms = declared_symbols()
    for name in ("vpmc_create", "vpmc_set_beam", "vpmc_set_range_shifter", "vpmc_set_aperture", "vpmc_dose", "vpmc_influence"):
        assert name in syms            # BASELINE.json north_star's call list


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2307_01416_b200 import build, binding
    path = build.build()
    lib = ctypes.CDLL(path)
    for name in declared_symbols():
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == declared_symbols()
    assert b"sm_100a" in ctypes.cast(lib.vpmc_version, ctypes.CFUNCTYPE(ctypes.c_char_p))()


def test_struct_mirrors_match_the_header_sizes():
    from paper_2307_01416_b200 import binding
    assert ctypes.sizeof(binding.Params) == 25 * 4
    assert ctypes.sizeof(binding.Tallies) == 6 * 8 + 8 * 8
    assert binding.STEP_DTYPE.itemsize == 80
    assert ctypes.sizeof(binding.Scenario) == 16
    assert binding.STATE_DTYPE.itemsize == 8 + 4 * 4 + 4 * 4 + 10 * 8
    assert binding.STATE_OUT_DTYPE.itemsize == 4 * 4 + 4 * 4 + 13 * 8


def test_default_params_without_gpu():
    from paper_2307_01416_b200 import binding
    p = binding.default_params()
    assert abs(p.alpha - 0.022) < 1e-9 and abs(p.p - 1.77) < 1e-7 and p.n_batches == 10 and p.flags == 7
    assert abs(p.brass_rsp - 5.523) < 1e-6


def test_compute_calls_fail_loudly_without_a_device():
    import numpy as np
    import torch
    if torch.cuda.is_available():
        return
    from paper_2307_01416_b200 import binding, workloads
    try:
        binding.Engine(workloads.small_water())
    except binding.VpmcError as e:
        assert e.code == binding.ERR_CUDA
    else:
        raise AssertionError("engine creation must fail without a CUDA device")
