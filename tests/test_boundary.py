"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/mg_toroidal.h declares; the binding covers all of them; no compute without a GPU."""
import ctypes
import os
import re

import pytest

from paper_2506_16676_b200 import binding, buildlib

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "mg_toroidal.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mg_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    buildlib.build()
    return ctypes.CDLL(buildlib.LIB_PATH)


def test_header_declares_the_survey_boundary():
    names = declared_symbols()
    for must in ("mg_setup", "mg_vcycle", "mg_solve", "mg_destroy", "mg_spmv", "mg_smooth", "mg_restrict",
                 "mg_prolong_add", "mg_coarse_solve", "mg_get_level", "mg_set_cheb_bounds", "mg_strerror"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in mg_toroidal.h but not exported"


def test_binding_covers_every_declared_symbol():
    assert sorted(binding.SYMBOLS) == declared_symbols()


def test_options_default_values():
    o = binding.options_default()
    assert (o.nu_pre, o.nu_post) == (2, 2)                      # "2 Chebyshev-PBJ sweeps", configs[0]
    assert (o.cheb_lo, o.cheb_hi, o.eig_iters) == (0.1, 1.1, 20)
    assert (o.coarse_mode, o.coarse_rtol, o.coarse_restart, o.coarse_maxit) == (0, 1e-10, 100, 20000)
    assert (o.restart, o.maxit) == (100, 400)
    assert binding.lib().mg_options_default(None) == binding.MG_EINVAL


def test_binding_struct_layouts_match_the_library(lib):
    lib.mg_sizeof_options.restype = ctypes.c_size_t
    lib.mg_sizeof_solve_info.restype = ctypes.c_size_t
    assert lib.mg_sizeof_options() == ctypes.sizeof(binding.mg_options)
    assert lib.mg_sizeof_solve_info() == ctypes.sizeof(binding.mg_solve_info)
    o = binding.options_default()
    assert (o.smoother, o.kernel_variant, o.use_graphs) == (0, 0, 1) and o.orth_eta == 0.25   # last fields land where C put them


def test_strerror_and_version():
    assert binding.strerror(0) == "ok"
    assert "singular" in binding.strerror(binding.MG_ESINGULAR)
    assert "sm_100a" in binding.version()


def test_no_cpu_fallback():
    """Without a CUDA device the product path fails loudly (it never routes through the oracle)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        binding.Solver(None, None, None, 6, 4, 4, 1)
    h = ctypes.c_void_p()
    buf = (ctypes.c_double * 64)()
    rc = binding.lib().mg_setup(ctypes.byref(h), ctypes.addressof(buf), ctypes.addressof(buf), ctypes.addressof(buf),
                                1, 1, 1, 1, None, None)
    assert rc == binding.MG_ECUDA and not h.value
    assert "no CPU fallback" in binding.strerror(rc)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2506_16676_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "mg_oracle" not in text, f
