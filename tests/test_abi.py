"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/c8opt.h declares; the binding's struct layouts match the header; calls that need a device fail
loudly (no CPU fallback) when there is none."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "c8opt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(c8opt_[a-z_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def c8():
    import __graft_entry__ as g
    g.build()
    import paper_2309_15861_b200 as c8
    return c8


def test_library_exports_every_declared_symbol(c8):
    names = _declared_functions()
    assert len(names) >= 9
    L = c8.lib()
    for n in names:
        assert hasattr(L, n), f"libc8opt.so does not export {n}"
    assert sorted(c8.EXPORTS) == names


def test_struct_layouts_match_header(c8):
    assert wl.SEGMENT_DTYPE.itemsize == 48                      # c8opt_segment
    assert c8.TALLY_DTYPE.itemsize == 24                        # c8opt_tally
    assert C.sizeof(c8._Layer) == 32
    assert C.sizeof(c8._AtmosphereDesc) == 8 + 8 * 32 + 24 + 8 + 32 + 8
    assert C.sizeof(c8._RunParams) == 8 + 8 + 6 * 8 + 8 + 8 + 8 + 8
    assert C.sizeof(c8._Output) == 5 * 8


def test_no_cpu_fallback(c8):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(c8.C8optError) as ei:
        c8.Context(wl.atmosphere_single_layer())
    assert ei.value.code == -2


def test_argument_errors_before_any_device_work(c8):
    L = c8.lib()
    assert L.c8opt_create_atmosphere(None, None) == -1
    d = c8._AtmosphereDesc()
    d.n_layers = 0
    h = C.c_void_p()
    assert L.c8opt_create_atmosphere(C.byref(d), C.byref(h)) == -1
    assert b"n_layers" in L.c8opt_last_error(None)
    assert L.c8opt_add_telescopes(None, None, 0) == -1
    assert L.c8opt_launch_count(None) == 0
    L.c8opt_destroy(None)


def test_product_does_not_import_oracle():
    """The product path never routes through the oracle."""
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2309_15861_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", txt, flags=re.M), f
                assert "liboracle" not in txt and "c8opt_oracle" not in txt, f
