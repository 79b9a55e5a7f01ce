"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol include/casgd.h
declares, and rejects bad arguments on the host before touching a device. No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_18463_b200 import build
    build.build()                                   # nvcc cross-compiles sm_100a without a GPU
    from paper_2606_18463_b200 import binding
    return binding.load()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "casgd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(casgd_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    from paper_2606_18463_b200 import binding
    declared = _declared_symbols()
    assert len(declared) >= 14
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/casgd.h but not exported by libcasgd.so"
    assert sorted(binding.EXPORTS) == declared


def test_version_names_the_arch(lib):
    assert b"sm_100a" in lib.casgd_version()


def test_library_holds_sm100a_code_only():
    import subprocess
    from paper_2606_18463_b200 import binding
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_bad_arguments_fail_on_the_host(lib):
    ctx = ctypes.c_void_p()
    dummy = ctypes.c_void_p(16)
    assert lib.casgd_init(None, dummy, 8, dummy, 4, 8, 0, None) == 1                    # out == NULL
    assert lib.casgd_init(ctypes.byref(ctx), None, 8, dummy, 4, 8, 0, None) == 1        # X == NULL
    assert lib.casgd_init(ctypes.byref(ctx), dummy, 8, None, 4, 8, 0, None) == 1        # y == NULL
    assert lib.casgd_init(ctypes.byref(ctx), dummy, 8, dummy, 0, 8, 0, None) == 1       # m < 1
    assert lib.casgd_init(ctypes.byref(ctx), dummy, 4, dummy, 4, 8, 0, None) == 1       # ldx < n
    assert lib.casgd_init(ctypes.byref(ctx), dummy, 8, dummy, 4, 8, 3, None) == 1       # unknown loss
    assert not ctx.value
    assert lib.casgd_outer_step(None, dummy, dummy, 1, 1, 0.1) == 1
    assert lib.casgd_loss(None, dummy, None) == 1
    assert lib.casgd_sync(None) == 1
    assert lib.casgd_launch_count(None) == 0
    lib.casgd_destroy(None)                                                             # allowed


def test_init_without_a_gpu_reports_an_error_not_a_crash(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present; the no-device path cannot be exercised")
    ctx = ctypes.c_void_p()
    dummy = ctypes.c_void_p(16)
    rc = lib.casgd_init(ctypes.byref(ctx), dummy, 8, dummy, 4, 8, 0, None)
    assert rc in (3, 4) and not ctx.value                                               # CASGD_ECUDA / CASGD_EARCH


def test_product_does_not_import_the_oracle():
    """The product path shares nothing with oracle/ (and oracle/ nothing with the product)."""
    pkg = os.path.join(ROOT, "paper_2606_18463_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "casgd_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2606_18463_b200\b", text, flags=re.M), f
            assert '#include "../' not in text
