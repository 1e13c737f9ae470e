"""CPU-only checks of the boundary: the C-ABI library builds (nvcc cross-compiles without a GPU), loads,
and exports every symbol include/apd.h declares; the binding has no fallback.  No compute call is made."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "apd.h")
PROBE_HEADER = os.path.join(ROOT, "include", "apd_probe.h")


def declared_functions(header=HEADER):
    src = open(header).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(apd_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2403_03571_b200 import build, binding
    build.build()
    return binding.load_library()


def test_header_declares_the_two_calls():
    names = declared_functions()
    for must in ("apd_assign", "apd_solve", "apd_create", "apd_destroy", "apd_last_error", "apd_default_opts",
                 "apd_assign_host", "apd_solve_host"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} is declared in include/apd.h but not exported"


def test_binding_lists_the_same_symbols():
    from paper_2403_03571_b200 import binding
    assert sorted(binding.EXPORTED_SYMBOLS) == declared_functions()


def test_every_header_under_include_is_covered():
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["apd.h", "apd_probe.h"]


def test_probe_library_exports_its_header_and_nothing_of_it_is_in_the_product(lib):
    """The FP32 microbenchmark is a bench-only library of its own (include/apd_probe.h)."""
    from paper_2403_03571_b200 import probe
    plib = probe.load_library()
    names = declared_functions(PROBE_HEADER)
    assert names == sorted(probe.EXPORTED_SYMBOLS) == ["apd_fp32_probe"]
    for name in names:
        assert hasattr(plib, name)
        assert not hasattr(lib, name), f"{name} must not be exported by the product library"


def test_struct_layouts_match_header(lib):
    from paper_2403_03571_b200 import binding
    assert ctypes.sizeof(binding.apd_grid) == 4 + 12 + 24 + 24
    assert ctypes.sizeof(binding.apd_opts) == 32
    o = binding.make_opts()
    assert (o.kernel, o.cull, o.lbfgs_history, o.max_iters, o.max_evals) == (0, 0, 10, 1000, 0)


def test_library_is_sm100a_only():
    from paper_2403_03571_b200 import build
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", build.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_no_fallback_when_library_missing(monkeypatch, tmp_path):
    from paper_2403_03571_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(ImportError):
        binding.load_library()


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2403_03571_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "apd_oracle" not in text, f
