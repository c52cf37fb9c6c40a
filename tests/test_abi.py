"""No-GPU checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/cyrsoxs.h declares; argument validation that needs no device."""
import ctypes as C
import os
import re

import pytest

from paper_2209_13121_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def test_header_symbols_are_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "cyrsoxs.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(cyrsoxs_[a-z_]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), f"{name} not exported"
    assert b"sm_100a" in lib.cyrsoxs_version()


def test_no_torch_types_in_signatures():
    hdr = open(os.path.join(ROOT, "include", "cyrsoxs.h")).read()
    assert "torch" not in hdr.lower().replace("pytorch", "") and "at::" not in hdr and "#include" not in hdr.split("extern")[1]


def test_create_rejects_bad_arguments_without_a_device(lib):
    h = C.c_void_p()
    # sizes: 4 <= Nx <= 2048, 2 <= Ny <= 2048, 1 <= Nz <= 2048, any length in between (DESIGN 3-A14)
    for args in [(0, 8, 8, 1, 1.0), (3, 8, 8, 1, 1.0), (8, 1, 8, 1, 1.0), (8, 8, 0, 1, 1.0), (8, 2049, 8, 1, 1.0), (8, 8, 4096, 1, 1.0), (8, 8, 8, 0, 1.0),
                 (8, 8, 8, 33, 1.0), (8, 8, 8, 1, 0.0), (8, 8, 8, 1, -1.0), (8192, 8, 8, 1, 1.0), (2, 8, 8, 1, 1.0)]:
        st = lib.cyrsoxs_create(*args, C.byref(h))
        assert st == binding.ERR_INVALID_ARG and not h.value, args
    assert lib.cyrsoxs_create(8, 8, 8, 1, 1.0, None) == binding.ERR_INVALID_ARG
    assert lib.cyrsoxs_last_error(None)          # static string, no crash
    lib.cyrsoxs_destroy(None)                     # NULL is fine


def test_null_context_is_rejected(lib):
    assert lib.cyrsoxs_set_angles(None, 0.0, 1.0, 2.0) == binding.ERR_INVALID_ARG
    assert lib.cyrsoxs_set_ewald(None, 0) == binding.ERR_INVALID_ARG
    assert lib.cyrsoxs_run(None, None, None) == binding.ERR_INVALID_ARG
    assert lib.cyrsoxs_num_angles(None) == 0


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2209_13121_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "cyrsoxs_oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "cyrsoxs_oracle.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_2209_13121_b200", osrc, flags=re.M)
    assert "kernels.cuh" not in osrc and "fft_core" not in osrc
