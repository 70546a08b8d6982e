"""CPU-side checks of the boundary: libgwc.so builds for sm_100a, loads, and exports every symbol that
include/gwc.h declares; the binding names the same entry points; the product package never touches oracle/."""
from __future__ import annotations

import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "gwc.h")


@pytest.fixture(scope="module")
def lib_path():
    from paper_2605_23538_b200 import build
    return build.build()


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gwc_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = _declared()
    for must in ("gwc_build_cosmo", "gwc_event_loglik", "gwc_selection_logxi", "gwc_total_loglik", "gwc_pack_events"):
        assert must in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in _declared():
        assert hasattr(lib, name), name


def test_binding_covers_the_header(lib_path):
    from paper_2605_23538_b200 import gwc
    assert sorted(gwc.EXPORTS) == _declared()
    gwc.load()
    for name in gwc.EXPORTS:
        if name in ("gwc_create", "gwc_destroy", "gwc_last_error"):
            continue
        assert hasattr(gwc.Context, name), name


def test_library_is_sm100a_only(lib_path):
    out = subprocess.run(["cuobjdump", "--list-elf", lib_path], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_context_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2605_23538_b200 import gwc
    with pytest.raises(RuntimeError):
        gwc.Context(0)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2605_23538_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "gwc_oracle" not in text, f
