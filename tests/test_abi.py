"""The C ABI without a GPU: libgdrr_b200.so loads, exports every function include/gdrr.h declares,
the Python binding binds exactly that set, and the host-only entry points behave (status codes,
never a crash or an exception across the ABI)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "gdrr.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"GDRR_API\s+[\w\s\*]+?\b(gdrr_\w+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for must in ("gdrr_create_volume", "gdrr_set_geometry", "gdrr_set_spectrum", "gdrr_project"):
        assert must in names
    assert len(names) >= 14


def test_library_exports_every_declared_function_and_binding_binds_them():
    import paper_1204_6367_b200 as g
    lib = ctypes.CDLL(g.LIBRARY_PATH)
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} is declared in include/gdrr.h but not exported"
    assert sorted(g.EXPORTS) == declared_functions()
    for name in g.EXPORTS:                              # a Python function of the same name wraps each
        assert callable(getattr(g, name)), name
    assert re.fullmatch(r"\d+\.\d+", g.gdrr_version())


def test_header_is_plain_c(tmp_path):
    """include/gdrr.h is a C header: it compiles alone as C99 (and as C++), no CUDA header needed."""
    import shutil
    import subprocess
    src = tmp_path / "t.c"
    src.write_text('#include "gdrr.h"\nint main(void) { const char* (*f)(void) = gdrr_version; (void)f; return 0; }\n')
    inc = os.path.join(ROOT, "include")
    subprocess.run([shutil.which("gcc") or "gcc", "-std=c99", "-pedantic", "-Wall", "-Werror", "-fsyntax-only", "-I", inc,
                    str(src)], check=True)
    subprocess.run([shutil.which("g++") or "g++", "-std=c++17", "-Wall", "-Werror", "-fsyntax-only", "-x", "c++", "-I", inc,
                    str(src)], check=True)


def test_host_only_calls_return_status_codes():
    import paper_1204_6367_b200 as g
    # workspace sizes are host arithmetic: 16 B per quad for the packed layout, VW floats per padded voxel otherwise
    n = g.gdrr_volume_workspace_bytes(32, 32, 32, 1, g.GDRR_LAYOUT_PACKED_QUAD)
    assert n >= 16 * 33 * 33 * 34 and n % 16 == 0
    assert g.gdrr_volume_workspace_bytes(30, 30, 30, 4, g.GDRR_LAYOUT_LINEAR) == 32 * 32 * 32 * 16
    with pytest.raises(g.GdrrError) as e:
        g.gdrr_volume_workspace_bytes(0, 4, 4, 1, g.GDRR_LAYOUT_LINEAR)
    assert e.value.code == g.GDRR_ERR_INVALID_ARG
    # more than four materials: one device volume per group of four (here 4 + 1 materials: float4 + float per voxel)
    assert g.gdrr_volume_workspace_bytes(30, 30, 30, 5, g.GDRR_LAYOUT_LINEAR) == 32 * 32 * 32 * (16 + 4)
    with pytest.raises(g.GdrrError) as e:
        g.gdrr_volume_workspace_bytes(8, 8, 8, g.GDRR_MAX_MATERIALS + 1, g.GDRR_LAYOUT_LINEAR)
    assert e.value.code == g.GDRR_ERR_UNSUPPORTED
    with pytest.raises(g.GdrrError) as e:
        g.gdrr_volume_workspace_bytes(8, 8, 8, 1, 7)
    assert e.value.code == g.GDRR_ERR_INVALID_ARG
    # NULL handles are rejected, not dereferenced
    assert g._lib.gdrr_set_method(None, 0) == g.GDRR_ERR_INVALID_ARG
    assert g._lib.gdrr_project(None, None, 0, 1, None, None, None, None) == g.GDRR_ERR_INVALID_ARG
    assert g.gdrr_kernel_launches(None) == 0


def test_no_cpu_fallback_without_a_device():
    """On a machine without a GPU, creating a context fails with a CUDA status (no CPU path)."""
    import torch
    import paper_1204_6367_b200 as g
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(g.GdrrError) as e:
        g.gdrr_create_context(0)
    assert e.value.code in (g.GDRR_ERR_CUDA, g.GDRR_ERR_INVALID_ARG)
    assert g.gdrr_last_error(None)
