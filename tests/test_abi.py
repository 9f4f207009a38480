"""CPU checks of the boundary: libgabsplat.so builds, loads, and exports every function that
include/gabsplat.h declares; the ctypes structs mirror the header; host-side size queries behave.
No compute call is made (there is no GPU here)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2508_05343_b200 import build
    path = build.build()
    return C.CDLL(path)


def declared_functions():
    src = open(os.path.join(ROOT, "include", "gabsplat.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gabsplat_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_four_calls():
    names = declared_functions()
    for n in ("gabsplat_preprocess", "gabsplat_bin_sort", "gabsplat_render_forward", "gabsplat_render_backward"):
        assert n in names


def test_every_declared_symbol_is_exported(lib):
    for n in declared_functions():
        assert hasattr(lib, n), n


def test_size_queries(lib):
    lib.gabsplat_packed_floats.restype = C.c_int32
    lib.gabsplat_sort_workspace_bytes.restype = C.c_uint64
    lib.gabsplat_sort_workspace_bytes.argtypes = [C.c_int32, C.c_uint64, C.c_int32, C.c_int32]
    lib.gabsplat_grad_workspace_bytes.restype = C.c_uint64
    assert [lib.gabsplat_packed_floats(k) for k in (0, 1, 2, 4, 8)] == [12, 16, 20, 24, 36]
    assert lib.gabsplat_packed_floats(9) == 0 and lib.gabsplat_packed_floats(-1) == 0
    a = lib.gabsplat_sort_workspace_bytes(1000, 10_000, 8000, 4000)
    b = lib.gabsplat_sort_workspace_bytes(1000, 20_000, 8000, 4000)
    assert b > a >= 10_000 * 8
    assert lib.gabsplat_grad_workspace_bytes(10, 4) >= 10 * 24 * 4
    assert lib.gabsplat_grad_workspace_bytes(10, 9) == 0


def test_struct_sizes_match_header():
    from paper_2508_05343_b200 import binding as gb
    assert C.sizeof(gb._Camera) == 4 * (2 + 4 + 12 + 1 + 3)
    assert C.sizeof(gb._Scene) == 16 + 7 * 8
    assert C.sizeof(gb._Projected) == 11 * 8
    assert C.sizeof(gb._Binning) == 10 * 8      # ... + tile_work_hint
    assert C.sizeof(gb._FwdOut) == 6 * 8        # ... + tile_work
    assert C.sizeof(gb._Grads) == 9 * 8


def test_create_fails_loudly_without_a_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2508_05343_b200 import binding as gb
    with pytest.raises(gb.GabsplatError):
        gb.Context(0)
    h = C.c_void_p()
    lib.gabsplat_create.argtypes = [C.POINTER(C.c_void_p), C.c_int32]
    assert lib.gabsplat_create(C.byref(h), 0) in (3, 4)
    assert not h.value
