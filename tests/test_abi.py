"""The C-ABI library builds, loads and exports every symbol include/pimd.h declares (CPU only:
no compute call is made here), and refuses to run without a CUDA device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2404_02628_b200 import binding, build

    build.build()
    return binding.load()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "pimd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pimd_[a-z0-9_]+)\s*\(", text)))


def test_header_and_binding_agree():
    from paper_2404_02628_b200 import binding

    assert declared_symbols() == sorted(binding.EXPORTED_SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.pimd_version()


def test_invalid_arguments_are_rejected_before_touching_the_device(lib):
    h = C.c_void_p()
    bad = [
        dict(N=0), dict(P=1), dict(d=4), dict(d=0), dict(beta=0.0), dict(beta=float("nan")), dict(s=0.0),
        dict(dt=0.0), dict(thermostat=3), dict(xi=float("inf")),
    ]
    base = dict(N=4, P=8, d=2, beta=2.0, omega=1.0, g=0.1, s=0.5, xi=1.0, dt=0.01, thermostat=1, seed=0)
    for kw in bad:
        a = dict(base, **kw)
        rc = lib.pimd_create(C.byref(h), a["N"], a["P"], a["d"], a["beta"], a["omega"], a["g"], a["s"], a["xi"], a["dt"],
                             a["thermostat"], a["seed"])
        assert rc == -1, kw
        assert not h.value
        assert lib.pimd_last_error(None)


def test_no_cpu_fallback(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p()
    rc = lib.pimd_create(C.byref(h), 4, 8, 2, 2.0, 1.0, 0.0, 0.5, 1.0, 0.01, 1, 0)
    assert rc == -3 and not h.value
    assert b"no CPU fallback" in lib.pimd_last_error(None)


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2404_02628_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "pimd_oracle" not in src, f
