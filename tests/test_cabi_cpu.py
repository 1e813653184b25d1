"""Host-side checks of the C-ABI library that need no GPU: it builds, loads, exports every symbol
declared in include/npfem.h, validates arguments and meshes, and refuses to run without a device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1911_03062_b200 import binding
from paper_1911_03062_b200.build import build
from workloads import icosahedron_cell_type, rbc_cell_type

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build()
    return binding.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "npfem.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(npfem_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared_symbols()
    assert len(names) >= 13
    assert sorted(binding.EXPORTED_SYMBOLS) == names
    for name in names:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.npfem_version()


def _create(lib, ct, type_of_cell, dt=0.1, precision=32, triangles=None, rest=None):
    rest = np.ascontiguousarray(ct.rest_positions if rest is None else rest, dtype=np.float64)
    tri = np.ascontiguousarray(ct.triangles if triangles is None else triangles, dtype=np.int32)
    arr = (binding._CellType * 1)()
    arr[0] = binding._CellType(rest.shape[0], tri.shape[0], rest.ctypes.data_as(C.POINTER(C.c_double)),
                               tri.ctypes.data_as(C.POINTER(C.c_int32)), binding._material_struct(ct.material))
    toc = np.ascontiguousarray(type_of_cell, dtype=np.int32)
    ctx = C.c_void_p()
    rc = lib.npfem_create(C.byref(ctx), arr, 1, toc.ctypes.data_as(C.POINTER(C.c_int32)), toc.shape[0],
                          dt, precision, 0, None)
    return rc, ctx, lib.npfem_last_error(None).decode()


def test_argument_validation(lib):
    ct = icosahedron_cell_type()
    rc, ctx, msg = _create(lib, ct, [0], precision=16)
    assert rc == -1 and not ctx.value and "precision" in msg
    rc, ctx, msg = _create(lib, ct, [0], dt=0.0)
    assert rc == -1 and "dt" in msg
    rc, ctx, msg = _create(lib, ct, [0, 1])
    assert rc == -1 and "type_of_cell[1]" in msg


def test_mesh_validation(lib):
    ct = icosahedron_cell_type()
    tri = ct.triangles.copy()
    rc, _, msg = _create(lib, ct, [0], triangles=tri[:-1])               # a hole
    assert rc == -2 and "not closed" in msg
    flipped = tri.copy()
    flipped[3] = flipped[3][::-1]                                         # one inconsistent face
    rc, _, msg = _create(lib, ct, [0], triangles=flipped)
    assert rc == -2 and "oriented" in msg
    rc, _, msg = _create(lib, ct, [0], triangles=tri[:, ::-1])            # inside-out
    assert rc == -2 and "counter-clockwise" in msg
    bad = tri.copy()
    bad[0, 0] = 99
    rc, _, msg = _create(lib, ct, [0], triangles=bad)
    assert rc == -2 and "out of range" in msg
    squashed = ct.rest_positions.copy()
    squashed[tri[0, 1]] = squashed[tri[0, 0]]
    rc, _, msg = _create(lib, ct, [0], rest=squashed)
    assert rc == -2 and "zero rest area" in msg


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    rc, ctx, msg = _create(lib, rbc_cell_type(2), [0, 0])
    assert rc == -3 and not ctx.value and "no CPU fallback" in msg
    with pytest.raises(binding.NpfemError):
        binding.Solver([rbc_cell_type(2)], [0], 0.1)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1911_03062_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".hpp", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("shares nothing with oracle/", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_1911_03062_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "(`paper_1911_03062_b200/`)", ""), f
