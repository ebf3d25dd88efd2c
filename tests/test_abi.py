"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol
include/mfdn_b200.h declares.  No compute call is made (no GPU here)."""
import ctypes
import os
import re

import pytest

from paper_1412_5989_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    return build.build()


def test_header_symbols_exported(libpath):
    header = open(os.path.join(ROOT, "include", "mfdn_b200.h")).read()
    declared = set(re.findall(r"\b(mfdn_[a-z0-9_]+)\s*\(", header))
    declared -= {"mfdn_status"}
    assert declared == set(binding.SYMBOLS)
    L = ctypes.CDLL(libpath)
    for name in declared:
        assert hasattr(L, name), name


def test_no_torch_types_in_abi():
    header = open(os.path.join(ROOT, "include", "mfdn_b200.h")).read()
    assert 'extern "C"' in header
    code = re.sub(r"/\*.*?\*/", "", header, flags=re.S)     # signatures only
    assert "torch" not in code.lower() and "at::" not in code and "std::" not in code


def test_sm100a_sass_present(libpath):
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_binding_argument_errors_without_gpu():
    # NULL out pointer -> MFDN_ERR_ARG before any CUDA call
    L = binding.lib()
    assert L.mfdn_orbitals_init(None, 0, 0, None, None, None, 0, None, None, None) == binding.MFDN_ERR_ARG
    assert L.mfdn_cg_build(None, None) == binding.MFDN_ERR_ARG
    assert L.mfdn_info(None, 0) == -1
    assert L.mfdn_last_error(None) == b"null context"


def test_product_path_does_not_touch_oracle():
    """The package must not import, link or read anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1412_5989_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, re.M), f
                assert "mscheme_oracle" not in src and "cg_exact" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1412_5989_b200.binding" not in src and "libmfdn" not in src and "csrc" not in src.replace("paper_1412_5989_b200/csrc", ""), f


def test_static_scratch_size_matches_binding():
    """include/mfdn_b200.h states the size of the static scratch array of mfdn_mscheme_static; the binding repeats it."""
    from paper_1412_5989_b200 import binding
    header = open(os.path.join(ROOT, "include", "mfdn_b200.h")).read()
    m = re.search(r"#define\s+MFDN_STATIC_SCRATCH_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", header)
    assert m, "MFDN_STATIC_SCRATCH_BYTES not found in the header"
    assert int(m.group(1)) << int(m.group(2)) == binding.MFDN_STATIC_SCRATCH_BYTES
    assert "mfdn_mscheme_static" in binding.SYMBOLS
