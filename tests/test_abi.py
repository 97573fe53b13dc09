"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol include/hashrender.h
declares; host-side argument validation that needs no GPU; the oracle is not reachable from the product package."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2409_10327_b200.build import build
    return build()


def test_header_symbols_exported(libpath):
    hdr = open(os.path.join(ROOT, "include", "hashrender.h")).read()
    declared = set(re.findall(r"\b(hashrender_[a-z_]+)\s*\(", hdr))
    assert {"hashrender_create", "hashrender_encode", "hashrender_decode", "hashrender_trace", "hashrender_shade",
            "hashrender_render_frame"} <= declared
    out = subprocess.check_output(["nm", "-D", "--defined-only", libpath], text=True)
    exported = set(re.findall(r"\bT (hashrender_[a-z_]+)", out))
    assert declared == exported, (declared ^ exported)
    from paper_2409_10327_b200.binding import EXPORTS
    assert set(EXPORTS) == declared
    lib = ctypes.CDLL(libpath)
    for name in declared:
        assert getattr(lib, name) is not None


def test_header_compiles_as_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "hashrender.h"\nint main(void){ hr_config c; hr_frame f; (void)c; (void)f; return HR_OK; }\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src), "-o",
                           str(tmp_path / "t.o")])


def test_null_handle_and_null_args_need_no_gpu(libpath):
    lib = ctypes.CDLL(libpath)
    lib.hashrender_last_error.restype = ctypes.c_char_p
    assert lib.hashrender_destroy(None) == 1
    assert lib.hashrender_encode(None, None, ctypes.c_uint64(4), None, None, None, None) == 1
    assert lib.hashrender_render_frame(None, None, None, None) == 1
    assert lib.hashrender_create(None, None, None, None, None) == 1
    assert lib.hashrender_last_error(None) == b"NULL handle"


def test_sass_is_sm100a_and_library_is_in_tree(libpath):
    assert os.path.dirname(libpath) == os.path.join(ROOT, "paper_2409_10327_b200")
    out = subprocess.check_output(["cuobjdump", "-lelf", libpath], text=True)
    assert "sm_100a" in out


def test_product_never_imports_oracle():
    """The product path must not route through the oracle (tier rule 3)."""
    pkg = os.path.join(ROOT, "paper_2409_10327_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "oracle" not in txt.replace("against the oracle", ""), f
    code = "import sys; import paper_2409_10327_b200; assert not any(m.startswith('oracle') for m in sys.modules)"
    subprocess.check_call([sys.executable, "-c", code], cwd=ROOT)


def test_binding_fails_loudly_without_library(tmp_path):
    from paper_2409_10327_b200 import binding
    old = binding._lib
    binding._lib = None
    try:
        with pytest.raises(ImportError):
            binding.load_library(str(tmp_path / "nope.so"))
    finally:
        binding._lib = old
