"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/fft3d.h declares; host-only calls behave; nothing computes without a GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import paper_2202_12756_b200 as m
    if not os.path.exists(m.binding.LIB_PATH):
        import __graft_entry__ as g
        g.build()
    return m.load_library()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "fft3d.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fft3d_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    import paper_2202_12756_b200 as m
    names = declared_functions()
    assert len(names) >= 12
    for nm in names:
        assert hasattr(lib, nm), "libfft3d.so does not export %s" % nm
    assert set(names) == set(m.binding.EXPORTS)


def test_host_only_calls(lib):
    import paper_2202_12756_b200 as m
    for n in (4, 64, 256, 1024, 1536, 2048, 768, 3072, 4096, 20, 640, 1280, 28, 896, 1792):
        assert m.supported_length(n)
    for n in (1, 5, 7, 1000, 8192, 9):
        assert not m.supported_length(n)
    assert "invalid" in m.strerror(1) and m.strerror(0) == "ok" and m.strerror(99)
    assert lib.fft3d_destroy(None) == 0
    assert lib.fft3d_workspace_bytes(None) == 0
    assert lib.fft3d_index(None, 0, 0, 0) == -1


def test_plan_validation_needs_no_gpu(lib):
    h = ctypes.c_void_p()
    assert lib.fft3d_plan(ctypes.byref(h), 64, 64, 63, 0, 1) == 2        # odd Nz
    assert lib.fft3d_plan(ctypes.byref(h), 64, 64, 64, 0, 3) == 1        # p does not divide
    assert lib.fft3d_plan(ctypes.byref(h), 64, 64, 64, 5, 1) == 1        # bad dtype
    assert lib.fft3d_plan(ctypes.byref(h), 1, 64, 64, 0, 1) == 1         # extent < 2
    assert lib.fft3d_plan(ctypes.byref(h), 44, 64, 64, 0, 1) == 2        # 44 = 11*4 unsupported (no radix 11)
    assert lib.fft3d_plan(None, 64, 64, 64, 0, 1) == 1


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2202_12756_b200 as m
    with pytest.raises(m.Fft3dError) as e:
        m.Plan(64, 64, 64)
    assert e.value.status == 4


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2202_12756_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), fn
                assert "oracle/" not in txt.replace("oracle/)", "") or fn == "inputs.py", fn
