"""CPU-side checks of the boundary: libwcras.so builds/loads, exports every symbol include/wcras.h declares,
and fails loudly (no CPU fallback) when no CUDA device is present.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

from paper_1011_3318_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def test_header_symbols_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "wcras.h")).read()
    declared = set(re.findall(r"\b(wcras_[a-z_A-Z0-9]+)\s*\(", hdr))
    assert declared, "no declarations found in include/wcras.h"
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), "libwcras.so does not export %s" % name


def test_no_torch_types_in_header():
    hdr = open(os.path.join(ROOT, "include", "wcras.h")).read()
    assert "torch" not in hdr.lower().replace("pytorch", "") and "at::" not in hdr
    assert 'extern "C"' in hdr


def test_info_struct_matches_header():
    hdr = open(os.path.join(ROOT, "include", "wcras.h")).read()
    body = hdr[hdr.index("typedef struct {"):hdr.index("} wcras_info;")]
    names = re.findall(r"\b(?:int|double)\s+([a-z_0-9]+);", body)
    assert names == [n for n, _ in binding.WcrasInfo._fields_]


def test_fails_loudly_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p(0)
    dims = (C.c_int * 4)(4, 4, 4, 4)
    dummy = (C.c_double * 8)()
    rc = lib.wcras_create(C.byref(h), dims, C.c_double(0.12), C.c_double(1.0), dummy, None)
    assert rc == binding.CUDA_ERROR and not h.value
    with pytest.raises(binding.WcrasError):
        binding.Context((4, 4, 4, 4), 0.12, 1.0, C.addressof(dummy))


def test_invalid_args(lib):
    h = C.c_void_p(0)
    assert lib.wcras_create(C.byref(h), None, C.c_double(0.12), C.c_double(1.0), None, None) == binding.INVALID_ARG
    assert lib.wcras_destroy(None) == binding.INVALID_ARG
    assert lib.wcras_apply_D(None, 32, None, None) == binding.INVALID_ARG
    lib.wcras_last_error.restype = C.c_char_p
    assert lib.wcras_last_error(None) == b"null ctx"


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1011_3318_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "wcoracle" not in src, f
    orc = open(os.path.join(ROOT, "oracle", "wcoracle.py")).read() + open(os.path.join(ROOT, "oracle", "wcoracle.c")).read()
    assert "import paper_1011_3318_b200" not in orc and "from paper_1011_3318_b200" not in orc and "csrc/" not in orc.replace("paper_1011_3318_b200/csrc/.", "")
