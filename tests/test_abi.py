"""CPU: the C-ABI library builds, loads and exports every symbol include/melt.h declares; the Python binding
lists the same names.  No compute call is made (there is no GPU here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_symbols(name="melt.h"):
    with open(os.path.join(ROOT, "include", name)) as fh:
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
    tsyms = _header_symbols("melt_test.h")           # the test aids live in their own header, outside the product API
    assert sorted(binding.TEST_SYMBOLS) == tsyms and not set(tsyms) & set(syms)
    for s in tsyms:
        assert hasattr(lib, s) and hasattr(binding, s), s


def test_frame_count_needs_no_gpu_and_matches_the_oracle():
    from oracle import melt_oracle as orc
    from paper_2606_01009_b200 import binding, sharding
    for n_fft, hop in ((400, 160), (401, 160), (1024, 256), (37, 7)):
        for length in (0, 1, n_fft // 2, n_fft // 2 + 1, n_fft - 1, n_fft, n_fft + hop - 1, n_fft + hop, 16000, 480000):
            for pad in (0, 1):
                for drop in (False, True):
                    want = orc.num_frames(length, n_fft, hop, pad, drop)
                    assert binding.melt_count_frames(length, n_fft, hop, pad, drop) == want, (n_fft, hop, length, pad, drop)
                    assert sharding.frames_of(length, n_fft, hop, bool(pad), drop) == want


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
