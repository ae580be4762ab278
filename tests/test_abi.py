"""CPU: the C-ABI library builds, loads and exports every symbol include/melt.h declares; the Python binding
lists the same names.  No compute call is made (there is no GPU here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_symbols():
    with open(os.path.join(ROOT, "include", "melt.h")) as fh:
        src = re.sub(r"/\*.*?\*/", "", fh.read(), flags=re.S)
    return sorted(set(re.findall(r"\b(melt_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    syms = _header_symbols()
    for need in ("melt_plan_create", "melt_forward", "melt_plan_destroy", "melt_forward_ragged", "melt_last_error"):
        assert need in syms


def test_library_exports_every_declared_symbol():
    from paper_2606_01009_b200 import binding, build
    lib = ctypes.CDLL(build.build())
    syms = _header_symbols()
    missing = [s for s in syms if not hasattr(lib, s)]
    assert not missing, missing
    assert sorted(binding.SYMBOLS) == syms
    for s in syms:                                   # the binding exposes the same names
        assert hasattr(binding, s), s


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_01009_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, f)) as fh:
                    txt = fh.read()
                assert "oracle" not in txt.lower() or f == "workloads.py", (f, "mentions the oracle")


def test_last_error_is_callable_without_a_gpu():
    from paper_2606_01009_b200 import binding
    assert isinstance(binding.melt_last_error(), str)
