"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports
every symbol include/helios.h declares; without a GPU the product fails loudly."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "helios.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(helios_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    syms = _declared_symbols()
    for name in ("helios_load_opacity", "helios_forward_batch", "helios_loglike_batch"):
        assert name in syms


def test_library_builds_and_exports_every_declared_symbol():
    from paper_1910_01070_b200 import build
    path = build.build_library()
    lib = ctypes.CDLL(path)
    for name in _declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/helios.h but not exported"


def test_binding_has_the_same_names():
    import paper_1910_01070_b200 as pkg
    for name in _declared_symbols():
        if name == "helios_last_error":
            continue            # surfaced through HeliosError
        assert hasattr(pkg, name), name


def test_no_oracle_or_cpu_fallback_in_the_product():
    pkg = os.path.join(ROOT, "paper_1910_01070_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "helios_oracle" not in src, f


def test_create_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_1910_01070_b200 as pkg
    with pytest.raises(pkg.HeliosError) as ei:
        pkg.helios_create(0, 0)
    assert ei.value.code == pkg.HELIOS_ECUDA
    with pytest.raises(RuntimeError):
        pkg.Helios(0)
