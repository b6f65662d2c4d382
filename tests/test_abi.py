"""The C-ABI library loads and exports every symbol include/lise.h declares (no compute calls, no GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "lise.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lise_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported():
    from paper_2009_00745_b200 import lise
    lib = lise.load()
    syms = declared_symbols()
    assert len(syms) >= 16
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in include/lise.h but not exported by liblise.so"
    assert set(lise.EXPORTS) == set(syms)


def test_no_torch_types_in_header_and_extern_c():
    text = open(os.path.join(ROOT, "include", "lise.h")).read()
    assert 'extern "C"' in text
    assert "torch" not in text.lower().replace("torch tensor", "") and "at::" not in text


def test_calls_without_gpu_fail_cleanly():
    """host-only entry points work without a device; lise_strerror covers all codes."""
    from paper_2009_00745_b200 import lise
    lib = lise.load()
    p = lise.default_params()
    assert abs(p.hbarc - 197.3269804) < 1e-12 and p.coulomb == 1
    for code in (0, -1, -2, -3, -4, -5, -99):
        assert len(lib.lise_strerror(code)) > 0
    assert lib.lise_default_params(None) == -1
    # an unknown line operator is refused before any CUDA call, and the message is kept for the calling thread
    import ctypes
    h = ctypes.c_void_p(1)
    assert lib.lise_create_with_line_operator(8, 8, 8, 1.0, 0.05, 1, 0, b"cufft", ctypes.byref(h)) == -1
    assert h.value is None and b"unknown line operator" in lib.lise_last_error(None)


def test_product_path_does_not_import_oracle():
    """the product package must never reach into oracle/ (parity claims depend on it)."""
    pkg = os.path.join(ROOT, "paper_2009_00745_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                if f.endswith(".py"):
                    assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                    assert "liblise_oracle" not in src, f
                else:
                    assert not re.search(r"#include[^\n]*oracle", src), f
