"""The C-ABI boundary without a GPU: libbifrost.so builds for sm_100a, loads, exports every symbol that
include/bifrost.h declares (and nothing in the binding is missing from the header), and the
entry points that need no device behave as documented.  No compute calls here."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "bifrost.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2210_02472_b200 import build
    from paper_2210_02472_b200.binding import load_library
    build.build()
    return load_library()


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)            # strip comments
    return sorted(set(re.findall(r"\b(bifrost_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for required in ("bifrost_acc", "bifrost_grad", "bifrost_dtmin", "bifrost_pn1", "bifrost_create",
                     "bifrost_destroy", "bifrost_strerror"):
        assert required in names


def test_library_exports_every_declared_symbol(lib):
    from paper_2210_02472_b200.binding import SYMBOLS
    names = declared_symbols()
    for name in names:
        assert hasattr(lib, name), f"{name} declared in include/bifrost.h but not exported"
    assert sorted(SYMBOLS) == names, "binding.SYMBOLS and include/bifrost.h disagree"


def test_header_compiles_as_plain_c(tmp_path):
    """`extern "C"`, plain pointers and sizes only: the header must be valid C99 on its own."""
    src = tmp_path / "t.c"
    src.write_text('#include "bifrost.h"\nint main(void) { return BIFROST_OK; }\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src),
                           "-o", str(tmp_path / "t.o")])


def test_library_is_sm100a_with_the_expected_kernels():
    from paper_2210_02472_b200.binding import LIB_PATH
    out = subprocess.run(["cuobjdump", "-lelf", LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out, out
    sass = subprocess.run(["cuobjdump", "-sass", LIB_PATH], capture_output=True, text=True).stdout
    assert "MUFU.RSQ64H" in sass and "DFMA" in sass and "LDGSTS" in sass


def test_error_paths_without_a_device(lib):
    import torch
    assert lib.bifrost_strerror(0) == b"ok"
    assert b"invalid" in lib.bifrost_strerror(-1)
    assert lib.bifrost_strerror(-99) == b"unknown error"
    h = ctypes.c_void_p()
    assert lib.bifrost_create(None, 0, 10) == -1                     # EINVAL: NULL out pointer
    assert lib.bifrost_create(ctypes.byref(h), 0, 0) == -1           # EINVAL: max_n <= 0
    assert lib.bifrost_create(ctypes.byref(h), 0, 1 << 31) == -1     # EINVAL: max_n >= 2^31
    assert lib.bifrost_destroy(None) == -1
    assert lib.bifrost_launch_count(None) == 0
    assert lib.bifrost_last_cuda_error(None) == b""
    assert lib.bifrost_acc(None, 1, None, None, None, 1, None, 1, 1.0, 0.0, None, None) == -1
    if not torch.cuda.is_available():
        assert lib.bifrost_create(ctypes.byref(h), 0, 10) == -2      # ECUDA: no device, no fallback
        assert not h.value
        from paper_2210_02472_b200.binding import BifrostError, Context
        with pytest.raises(BifrostError):
            Context(10)
