"""CPU-only checks of the boundary: libfenc.so builds, loads, and exports every symbol include/fenc.h declares
(no compute calls without a GPU); the product path fails loudly without a CUDA device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    text = open(os.path.join(ROOT, "include", "fenc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fenc_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2606_16359_b200 import SYMBOLS, load_library
    lib = load_library()
    declared = header_symbols()
    assert declared == sorted(SYMBOLS)
    for name in declared:
        assert isinstance(getattr(lib, name), ctypes._CFuncPtr), name


def test_struct_layouts_match_header():
    from paper_2606_16359_b200 import ConvDesc, FcDesc, Layout, ParamsDesc
    assert ctypes.sizeof(ConvDesc) == 14 * 4
    assert ctypes.sizeof(FcDesc) == 10 * 4
    assert ctypes.sizeof(Layout) == 22 * 4 + 2 * 8 + 512 * 4
    assert ParamsDesc.log2_scale.offset == 32 and ParamsDesc.q_override.offset == 40


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2606_16359_b200 as fenc
    with pytest.raises(fenc.FencError):
        fenc.Context(6, 4, 30, 2, 31, 2, 25)
    # and the C entry point itself refuses without a device
    lib = fenc.load_library()
    d = fenc.ParamsDesc()
    d.log2N, d.n_q, d.q_bits, d.n_p, d.p_bits, d.dnum, d.log2_scale = 6, 4, 30, 2, 31, 2, 25.0
    h = ctypes.c_void_p()
    assert lib.fenc_params_init(ctypes.byref(d), ctypes.byref(h)) == 8  # FENC_ERR_DEVICE


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_16359_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "fenc_oracle" not in src, f
