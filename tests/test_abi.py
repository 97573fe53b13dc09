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


def test_binding_rejects_wrong_dtype_placement_and_alignment():
    """The binding marshals raw pointers, so it must refuse what the C side cannot see: a float64 array, a host array handed to a
    device entry point (or the reverse), a misaligned pdf buffer."""
    import numpy as np
    from paper_2409_10327_b200 import binding as B
    a32, a64 = np.zeros((4, 3), np.float32), np.zeros((4, 3), np.float64)
    assert B._arg(None, "x") is None
    assert B._arg(a32, "x", "f32", "host").value == a32.ctypes.data
    with pytest.raises(TypeError):
        B._arg(a64, "x", "f32", "host")
    with pytest.raises(TypeError):
        B._arg(a32, "x", "f32", "device")                     # a host array is not a device pointer
    with pytest.raises(ValueError):
        B._arg(np.zeros(9, np.float32)[1:], "pdf", "f32", "host", align=8)
    import torch
    t = torch.zeros((4, 3))
    assert B._arg(t, "x", "f32", "host").value == t.data_ptr()
    with pytest.raises(TypeError):
        B._arg(t.double(), "x", "f32", "host")
    with pytest.raises(TypeError):
        B.DirSet(a32.reshape(1, 4, 3), a64[:, 0].reshape(1, 4)).c("host")
    d = B.DirSet(np.zeros(40, np.float32), np.zeros(13, np.float32), S=3, point_stride=12).c("host")
    assert d.S == 3 and d.point_stride == 12
