"""The C-ABI library loads and exports every symbol include/mbs.h declares (no compute calls: no GPU here)."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2410_02395_b200 import build
    return build.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "mbs.h")).read()
    return sorted(set(re.findall(r"MBS_API[^;(]*?\b(mbs_\w+)\s*\(", text)))


def test_header_declares_the_boundary():
    names = declared_symbols()
    for required in ("mbs_create", "mbs_set_potential", "mbs_apply_operator", "mbs_solve", "mbs_destroy"):
        assert required in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in declared_symbols():
        assert hasattr(lib, name), name
    from paper_2410_02395_b200 import binding
    assert sorted(binding.DECLARED_SYMBOLS) == declared_symbols()


def test_fft_plan_table(lib_path):
    lib = ctypes.CDLL(lib_path)
    lib.mbs_fft_supported.argtypes = [ctypes.c_int64]
    for M in (128, 256, 320, 512, 630, 1260):   # the BASELINE.json configs and the paper's own 1260-voxel axis
        assert lib.mbs_fft_supported(M) == 1
    for M in (0, 7, 88, 1250):
        assert lib.mbs_fft_supported(M) == 0


def test_create_rejects_bad_arguments_without_gpu(lib_path):
    """Argument validation happens before any CUDA call."""
    from paper_2410_02395_b200 import binding as B
    with pytest.raises(B.MBSError) as e:
        B.mbs_create((100,), 0.25, 1.0, (4,), (3,), None, 8)
    assert e.value.status == B.MBS_ERR_INVALID_ARG
    with pytest.raises(B.MBSError) as e:
        B.mbs_create((176,), 0.25, 1.0, (4,), (2,), None, 8)
    assert e.value.status == B.MBS_ERR_UNSUPPORTED_SIZE
    assert "88" in str(e.value)
    with pytest.raises(B.MBSError) as e:                      # 2^31 voxels: one more than the kernels' 32-bit counters hold
        B.mbs_create((2048, 1024, 1024), 0.25, 1.0, (4, 4, 4), (2, 2, 2), None, 8)
    assert e.value.status == B.MBS_ERR_INVALID_ARG and "2^31" in str(e.value)


def test_header_compiles_as_c():
    src = '#include "mbs.h"\nint main(void){ mbs_info i; (void)i; return MBS_OK; }\n'
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-x", "c", "-",
                        "-fsyntax-only"], input=src, text=True, capture_output=True)
    assert r.returncode == 0, r.stderr


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2410_02395_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, re.M), f
    otext = open(os.path.join(ROOT, "oracle", "mbs_oracle.py")).read()
    assert "paper_2410_02395_b200" not in re.sub(r'""".*?"""', "", otext, flags=re.S)
