"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/pyslice_b200.h declares; the binding refuses to run without a GPU (no CPU fallback)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2602_10064_b200 import build, binding
    build.build()
    return binding.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "pyslice_b200.h")).read()
    return sorted(set(re.findall(r"PS_API[^;(]*?\b(ps_\w+)\s*\(", text)))


def test_header_declares_the_calls_of_the_hot_path():
    syms = declared_symbols()
    for must in ("ps_build_slices", "ps_multislice", "ps_tacaw", "ps_spectrum_image", "ps_sdp", "ps_make_incident",
                 "ps_tacaw_begin", "ps_tacaw_add", "ps_tacaw_finish", "ps_dispersion", "ps_qbin"):
        assert must in syms


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in the header but not exported"


def test_binding_covers_every_declared_symbol():
    from paper_2602_10064_b200 import binding
    assert sorted(binding.exported_symbols()) == declared_symbols()


def test_version_and_null_handling(lib):
    assert b"sm_100a" in lib.ps_version()
    assert lib.ps_launch_count(None) == 0
    lib.ps_destroy(None)                                      # must be a no-op


def test_no_cpu_fallback():
    import torch
    import paper_2602_10064_b200 as ps
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        ps.Context()


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2602_10064_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f"{f} mentions the oracle"
