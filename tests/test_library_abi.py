"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/implicit_filter.h declares; argument errors are reported without a GPU.  No compute calls here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2404_07398_b200 import build, binding
    build.build()
    return binding.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "implicit_filter.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(if_[a-z_]+)\s*\(", text)))


def test_header_symbols_all_exported(lib):
    from paper_2404_07398_b200 import EXPORTS
    names = declared_symbols()
    assert set(names) == set(EXPORTS), (names, EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None


def test_strerror_and_launch_count(lib):
    assert lib.if_strerror(0) == b"ok"
    assert b"degenerate" in lib.if_strerror(-3)
    assert lib.if_launch_count() >= 0


def test_argument_errors_without_gpu(lib):
    from paper_2404_07398_b200.binding import IF_EINVAL
    out = C.c_void_p()
    coords = np.zeros((3, 2))
    tri = np.zeros((1, 3), dtype=np.int32)
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    assert lib.if_prepare(None, 2, 3, p(tri), 1, None, None, C.byref(out)) == IF_EINVAL
    assert lib.if_prepare(p(coords), 4, 3, p(tri), 1, None, None, C.byref(out)) == IF_EINVAL
    assert lib.if_prepare(p(coords), 2, 3, p(tri), 0, None, None, C.byref(out)) == IF_EINVAL
    n = C.c_size_t()
    assert lib.if_workspace_bytes(None, 1, 16, C.byref(n)) == IF_EINVAL
    assert lib.if_mesh_info(None, None, None, None, None, None) == IF_EINVAL
    lib.if_destroy(None)


def test_no_device_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2404_07398_b200 import ImplicitFilterError, if_prepare
    from workloads import grid_mesh
    m = grid_mesh(4)
    with pytest.raises(ImplicitFilterError):
        if_prepare(m.coords, m.tri, m.period)
    # the C entry point itself reports IF_ECUDA, never a CPU result
    out = C.c_void_p()
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    rc = lib.if_prepare(p(m.coords), 2, m.n_vert, p(m.tri), m.n_tri, p(m.period), None, C.byref(out))
    assert rc == -6 and not out.value
