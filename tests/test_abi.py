"""The C-ABI library loads and exports every symbol include/paraiso_hydro.h declares (no compute calls, no GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "paraiso_hydro.h")


@pytest.fixture(scope="module")
def lib():
    from paper_1204_4779_b200 import binding, build

    build.build()
    return binding.load_library()


def declared_symbols():
    text = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)
    return sorted(set(re.findall(r"\b(paraiso_hydro_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = declared_symbols()
    for must in ("create", "set_state", "cfl_dt", "step", "get_state", "destroy"):
        assert f"paraiso_hydro_{must}" in names


def test_library_exports_every_declared_symbol(lib):
    from paper_1204_4779_b200 import binding

    names = declared_symbols()
    assert len(names) >= 16
    raw = ctypes.CDLL(binding.LIB_PATH)
    for name in names:
        assert hasattr(raw, name), name
    assert set(binding.SIGNATURES) == set(names)


def test_library_exports_the_wave_example(lib):
    """include/paraiso_wave.h (the paper's linear-wave example, §2.3) is exported by the same library."""
    from paper_1204_4779_b200 import binding

    text = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "paraiso_wave.h")).read(), flags=re.S)
    names = sorted(set(re.findall(r"\b(paraiso_wave_[a-z_]+)\s*\(", text)))
    assert names == sorted(binding.WAVE_SIGNATURES) and len(names) == 6
    raw = ctypes.CDLL(binding.LIB_PATH)
    for name in names:
        assert hasattr(raw, name), name
    h = ctypes.c_void_p()
    assert lib.paraiso_wave_create(ctypes.byref(h), 2, 3.43) == binding.PARAISO_EINVAL      # n < 3
    assert lib.paraiso_wave_create(ctypes.byref(h), 64, 0.0) == binding.PARAISO_EINVAL      # c <= 0
    assert lib.paraiso_wave_destroy(None) == binding.PARAISO_OK


def test_probe_library_exports_every_declared_symbol(lib):
    """include/paraiso_hydro_probe.h: the test / measurement probes live in a library of their own."""
    from paper_1204_4779_b200 import binding

    text = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "paraiso_hydro_probe.h")).read(), flags=re.S)
    names = sorted(set(re.findall(r"\b(paraiso_probe_[a-z_]+)\s*\(", text)))
    assert names == sorted(binding.PROBE_SIGNATURES)
    raw = ctypes.CDLL(binding.PROBE_PATH)
    for name in names:
        assert hasattr(raw, name), name
    product = ctypes.CDLL(binding.LIB_PATH)
    for name in names:
        assert not hasattr(product, name), "probes must not be exported by the product library"
    assert not hasattr(product, "paraiso_hydro_debug_arith")


def test_version_and_error_strings_need_no_device(lib):
    assert lib.paraiso_hydro_version().decode().startswith("paraiso_hydro")
    assert isinstance(lib.paraiso_hydro_last_error(None), bytes)


def test_create_rejects_bad_arguments_before_touching_the_device(lib):
    from paper_1204_4779_b200 import binding

    h = ctypes.c_void_p()
    n = (ctypes.c_int64 * 3)(16, 16, 16)
    e = (ctypes.c_double * 3)(1.0, 1.0, 1.0)
    f = lib.paraiso_hydro_create
    assert f(ctypes.byref(h), 4, n, e, 1.4, 0) == binding.PARAISO_EINVAL
    assert f(ctypes.byref(h), 0, n, e, 1.4, 0) == binding.PARAISO_EINVAL
    assert f(ctypes.byref(h), 2, n, e, 1.0, 0) == binding.PARAISO_EINVAL
    assert f(ctypes.byref(h), 2, n, e, 1.4, 7) == binding.PARAISO_EINVAL
    n3 = (ctypes.c_int64 * 3)(16, 3, 16)
    assert f(ctypes.byref(h), 2, n3, e, 1.4, 0) == binding.PARAISO_EINVAL
    e0 = (ctypes.c_double * 3)(1.0, 0.0, 1.0)
    assert f(ctypes.byref(h), 2, n, e0, 1.4, 0) == binding.PARAISO_EINVAL
    assert f(None, 2, n, e, 1.4, 0) == binding.PARAISO_EINVAL
    assert not h.value
    assert b"create" in lib.paraiso_hydro_last_error(None)
    assert lib.paraiso_hydro_destroy(None) == binding.PARAISO_OK


def test_no_cpu_fallback_without_a_device(lib):
    """On a box without a GPU the product path must fail loudly (PARAISO_ECUDA), never compute on the CPU."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1204_4779_b200 import binding

    with pytest.raises(binding.ParaisoError) as ei:
        binding.ParaisoHydro((16, 16), (1.0, 1.0), 1.4, "float32")
    assert ei.value.code == binding.PARAISO_ECUDA
    assert "no CPU fallback" in str(ei.value)


def test_product_path_never_imports_the_oracle():
    """Neither side imports, includes or links the other (only inputs.py, which holds no arithmetic, serves both)."""
    imp = re.compile(r"^\s*(import|from)\s+oracle\b", re.M)
    pkg = os.path.join(ROOT, "paper_1204_4779_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not imp.search(text), f
                assert "euler_oracle" not in text and "liboracle" not in text, f
    odir = os.path.join(ROOT, "oracle")
    for f in os.listdir(odir):
        if f.endswith((".py", ".cpp", ".h", ".c")):
            text = open(os.path.join(odir, f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1204_4779_b200\b", text, re.M), f
            assert not re.search(r"#include\s+\"[^\"]*(csrc|paraiso_hydro)", text), f
            assert "libparaiso_hydro" not in text, f
