"""CPU-side checks of the C-ABI library: it builds, loads without a GPU, exports every symbol
include/pic_b200.h declares, and its host-only entry points validate arguments."""
import ctypes as C
import os
import re

import pytest

from paper_2110_08650_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "pic_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pic_[a-z_]+)\s*\(", src)))


def test_header_and_binding_agree():
    assert _declared_symbols() == sorted(binding.SYMBOLS)


def test_library_loads_and_exports_every_symbol():
    L = binding.load_library()
    for name in _declared_symbols():
        assert hasattr(L, name), name


def test_workspace_bytes_validation_and_size():
    # config 2: 33.5M particles -> 32 B record + u32 id per slot, two pools, ~2.7 GB
    n = 128 ** 3 * 16
    b = binding.workspace_bytes((128, 128, 128), (8, 8, 4), 2, n)
    assert 2 * 36 * n < b < 3.3 * 36 * n      # two pools of 36 B slots + grids (two field buffers) + bookkeeping
    with pytest.raises(binding.PicError) as e:
        binding.workspace_bytes((100, 128, 128), (8, 8, 4), 2, n)
    assert e.value.code == binding.PIC_EINVAL
    with pytest.raises(binding.PicError):
        binding.workspace_bytes((128, 128, 128), (4, 4, 4), 2, n)
    with pytest.raises(binding.PicError):
        binding.workspace_bytes((128, 128, 128), (8, 8, 4), 4, n)
    # config 5 (two pools, 537 M particles) fits comfortably in 180 GB
    assert binding.workspace_bytes((512, 512, 256), (8, 8, 4), 3, 512 * 512 * 256 * 8) < 90e9


def test_create_rejects_bad_arguments_without_touching_the_gpu():
    L = binding.load_library()
    h = C.c_void_p(None)
    grid = (C.c_int32 * 3)(16, 16, 16)
    sc = (C.c_int32 * 3)(8, 8, 4)
    cell = (C.c_double * 3)(1.0, 1.0, 1.0)
    assert L.pic_create(C.byref(h), grid, cell, 1.5, sc, 1, 10, C.c_void_p(256), 1 << 30, None) == binding.PIC_EINVAL
    assert L.pic_create(C.byref(h), grid, cell, 0.5, sc, 1, 10, None, 1 << 30, None) == binding.PIC_EINVAL
    assert L.pic_create(C.byref(h), grid, cell, 0.5, sc, 1, 10, C.c_void_p(256), 16, None) == binding.PIC_ENOMEM
    assert b"workspace" in L.pic_last_error(None)
    assert not h.value


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2110_08650_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "pic_oracle" not in text, f
