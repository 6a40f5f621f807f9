"""CPU-side checks of the boundary: libpct.so builds for sm_100a, loads, and exports every symbol that
include/pct.h declares.  No compute call is made (there is no GPU here)."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1802_01070_b200 import build
    return build.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "pct.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pct_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    syms = declared_symbols()
    for name in ("pct_generate_mlp", "pct_solve", "pct_forward_project", "pct_column_counts", "pct_paths_decode",
                 "pct_create", "pct_destroy", "pct_reconstruct_host"):
        assert name in syms


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in declared_symbols():
        assert hasattr(lib, name), name
    from paper_1802_01070_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()
    binding.load_library()


def test_library_is_sm100a_only(lib_path):
    out = subprocess.run(["cuobjdump", "-lelf", lib_path], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_invalid_arguments_are_reported_without_a_gpu(lib_path):
    from paper_1802_01070_b200 import binding
    L = binding.load_library()
    out = ctypes.c_void_p()
    assert L.pct_create(None, None, 0, ctypes.byref(out)) == binding.E_INVALID_ARG
    assert L.pct_create(None, None, 0, None) == binding.E_INVALID_ARG
    g = binding.Geometry(0, 4, 4, 1.0, (ctypes.c_double * 3)(0, 0, 0))
    p = binding.MlpParams((ctypes.c_double * 6)(1e-6, 0, 0, 0, 0, 0), 100.0, 361.0, 0.038, 0.5, 1e-9, 2048)
    assert L.pct_create(ctypes.byref(g), ctypes.byref(p), 0, ctypes.byref(out)) == binding.E_INVALID_ARG
    assert L.pct_paths_info(None, None) == binding.E_INVALID_ARG
    L.pct_destroy(None)
    L.pct_paths_free(None)


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1802_01070_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("CPU oracle", "").replace("oracle/", "").replace("oracle's", "").replace("oracle tests", "").replace("oracle and", ""), f
                assert "pcto" not in text, f


def test_oracle_and_synth_are_independent_of_the_product():
    """The oracle imports nothing of the product; the shared input generator (synth/) holds no method arithmetic and
    imports neither side."""
    for d in ("oracle", "synth"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, d)):
            for f in files:
                if f.endswith((".py", ".cpp", ".h", ".c")):
                    text = open(os.path.join(dirpath, f)).read()
                    assert not re.search(r"(import|from)\s+paper_1802_01070_b200|#include\s*[\"<]pct[._]|libpct\.so|csrc/", text), f
                    if d == "synth":
                        assert "pcto" not in text and "import oracle" not in text and "from oracle" not in text, f
