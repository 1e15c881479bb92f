"""CPU-side checks of the boundary: libpimpc.so builds, loads, exports every symbol that
include/pimpc.h declares, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2601_14414_b200 import build, pimpc
    build.build()
    return pimpc.load()


def _declared():
    src = open(os.path.join(ROOT, "include", "pimpc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pimpc_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported_and_bound(lib):
    from paper_2601_14414_b200 import pimpc
    names = _declared()
    assert {"pimpc_create", "pimpc_set_stage", "pimpc_solve", "pimpc_get"} <= set(names)   # BASELINE.json north_star
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/pimpc.h but not exported"
        assert n in pimpc.SYMBOLS, f"{n} has no ctypes signature in the binding"
    assert set(pimpc.SYMBOLS) == set(names)


def test_struct_layouts_match_header(lib):
    from paper_2601_14414_b200 import pimpc
    assert ctypes.sizeof(pimpc.pimpc_result) == 48 and pimpc.RESULT_DTYPE.itemsize == 48
    for f, _ in pimpc.pimpc_result._fields_:
        assert getattr(pimpc.pimpc_result, f).offset == pimpc.RESULT_DTYPE.fields[f][1]
    assert ctypes.sizeof(pimpc.pimpc_tune) == 32
    o = pimpc.pimpc_opts()
    ctypes.memset(ctypes.byref(o), 0xFF, ctypes.sizeof(o))
    lib.pimpc_default_opts(ctypes.byref(o))
    assert (o.dtype, o.engine, o.rho, o.eta, o.c0, o.history) == (0, 0, 1.0, 0.999, 1.0, 0)
    assert o.workspace is None and o.workspace_bytes == 0
    assert all(getattr(o.tune, f) == 0 for f, _ in pimpc.pimpc_tune._fields_)
    # the header's struct members, in order, are the binding's fields
    src = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "pimpc.h")).read(), flags=re.S)
    for cname, cls in (("pimpc_tune", pimpc.pimpc_tune), ("pimpc_opts", pimpc.pimpc_opts), ("pimpc_result", pimpc.pimpc_result),
                       ("pimpc_info", pimpc.pimpc_info), ("pimpc_peaks", pimpc.pimpc_peaks)):
        body = re.search(r"typedef struct \{([^{}]*)\} " + cname + ";", src).group(1)
        names = [re.search(r"(\w+)\s*$", part).group(1) for decl in body.split(";") if decl.strip() for part in decl.split(",")]
        assert names == [f for f, _ in cls._fields_], (cname, names)
    assert b"sm_100a" in lib.pimpc_version()


def test_workspace_bytes_and_argument_validation(lib):
    from paper_2601_14414_b200 import pimpc
    o = pimpc.pimpc_opts(); lib.pimpc_default_opts(ctypes.byref(o))
    assert lib.pimpc_workspace_bytes(0, 1, 1, 1, ctypes.byref(o)) == 0
    assert lib.pimpc_workspace_bytes(100, 61, 1, 1, ctypes.byref(o)) == 0        # nx + nu > 160
    assert lib.pimpc_workspace_bytes(100, 30, 1, 1, ctypes.byref(o)) > 0         # the paper's largest Table-I shape
    assert lib.pimpc_workspace_bytes(2, 1, 3, 70000, ctypes.byref(o)) == 0       # batch > 65535
    w64 = lib.pimpc_workspace_bytes(12, 4, 50, 4096, ctypes.byref(o))
    o.dtype = pimpc.F32
    w32 = lib.pimpc_workspace_bytes(12, 4, 50, 4096, ctypes.byref(o))
    # A, B, H, M and three state buffers dominate: (144+48+256+16+3*88+16+4) floats per stage
    per_stage = 144 + 48 + 256 + 16 + 3 * 88 + 16 + 4
    assert w32 >= 4096 * 50 * per_stage * 4 and w32 < 1.2 * 4096 * 50 * per_stage * 4
    assert abs(w64 / w32 - 2.0) < 0.05
    h = ctypes.c_void_p()
    assert lib.pimpc_create(ctypes.byref(h), 0, 1, 1, 1, None) == pimpc.EINVAL
    assert lib.pimpc_create(None, 1, 1, 1, 1, None) == pimpc.EINVAL
    assert b"positive" in lib.pimpc_last_error(None) or b"NULL" in lib.pimpc_last_error(None)


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2601_14414_b200 import pimpc
    with pytest.raises(pimpc.PimpcError) as e:
        pimpc.Solver(2, 1, 3, 1)
    assert e.value.code == pimpc.ECUDA and "no CPU fallback" in str(e.value)


def test_product_path_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package may import, link or run it, and the
    oracle imports nothing from the package and includes none of its headers."""
    imp = re.compile(r"^\s*(from|import)\s+(\S+)", re.M)
    pkg = os.path.join(ROOT, "paper_2601_14414_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            txt = open(os.path.join(dirpath, f), errors="ignore").read() if f.endswith((".py", ".cu", ".h")) else ""
            if f.endswith(".py"):
                assert not [m for m in imp.findall(txt) if m[1].split(".")[0] == "oracle"], f
            assert "pimpc_oracle" not in txt and "libpimpc_oracle" not in txt, f
    for f in ("pimpc_oracle.py", "pimpc_oracle.c"):
        txt = open(os.path.join(ROOT, "oracle", f)).read()
        assert not [m for m in imp.findall(txt) if m[1].startswith("paper_2601_14414_b200")], f
        assert not re.search(r'#include\s+"[^"]*pimpc(_internal)?\.h"', txt) and "libpimpc.so" not in txt, f
