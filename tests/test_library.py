"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/gecc.h declares.  No compute call is made (there is no GPU here)."""
import ctypes
import os
import re
import shutil

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "gecc.h")


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gecc_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2508_04355_b200 import build
    if not os.path.exists(build.LIB):
        if shutil.which("nvcc") is None and not os.path.exists("/usr/local/cuda/bin/nvcc"):
            pytest.skip("no nvcc and no prebuilt library")
        build.build()
    return build.LIB


def test_header_declares_the_three_named_entry_points():
    syms = declared_symbols()
    for name in ("gecc_encode", "gecc_matmul_protected", "gecc_decode_correct"):
        assert name in syms


def test_library_loads_and_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in declared_symbols():
        assert hasattr(lib, name), name
    lib.gecc_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.gecc_version()


def test_binding_lists_the_same_symbols(lib_path):
    from paper_2508_04355_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()
    binding.load()


def test_workspace_bytes_is_host_only_and_monotone(lib_path):
    from paper_2508_04355_b200 import binding
    a = binding.gecc_workspace_bytes(binding.GECC_BF16, 1024, 1024, 1024)
    b = binding.gecc_workspace_bytes(binding.GECC_BF16, 4096, 4096, 4096)
    assert 0 < a < b
    assert binding.gecc_workspace_bytes(5, 64, 64, 64) == 0


def test_report_struct_layout_matches_the_header():
    from paper_2508_04355_b200 import binding
    # verdict, n_found, n_row_flags, n_col_flags (4 x int32) + 4 + 4 doubles + 8 x (4 int32 + double)
    assert ctypes.sizeof(binding.GeccReport) == 16 + 64 + 8 * 24
    assert ctypes.sizeof(binding.GeccFault) == 16


def test_sass_contains_the_blackwell_instructions(lib_path):
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("no cuobjdump")
    import subprocess
    sass = subprocess.run([cuobjdump, "-sass", lib_path], capture_output=True, text=True).stdout
    for mnemonic in ("UTCHMMA", "UTMALDG", "LDTM"):      # tcgen05.mma, TMA load, tcgen05.ld
        assert mnemonic in sass, mnemonic
