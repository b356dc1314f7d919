"""CPU-only checks of the boundary: librsdft.so builds for sm_100a, loads, exports every symbol
include/rsdft.h declares, and rejects bad arguments before touching the device.  No compute
calls are made here (there is no GPU on this box and no CPU fallback in the product)."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2512_04447_b200 import build, rsdft
    build.build()
    return rsdft.load()


def test_header_symbols_are_exported(lib):
    from paper_2512_04447_b200 import rsdft
    header = open(os.path.join(ROOT, "include", "rsdft.h")).read()
    declared = sorted(set(re.findall(r"\b(rsdft_[a-z_0-9]+)\s*\(", header)))
    assert declared, "no declarations parsed"
    assert sorted(rsdft.SYMBOLS) == declared
    for name in declared:
        assert hasattr(lib, name), name
    out = subprocess.check_output(["nm", "-D", "--defined-only", rsdft.LIB_PATH]).decode()
    exported = set(re.findall(r" T (rsdft_[a-z_0-9]+)", out))
    assert exported == set(declared)


def test_library_holds_sm100a_code_only():
    from paper_2512_04447_b200 import rsdft
    out = subprocess.check_output(["/usr/local/cuda/bin/cuobjdump", "--list-elf", rsdft.LIB_PATH]).decode()
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "rsdft.h"\nint main(void){ rsdft_grid_t g; (void)g; return RSDFT_OK; }\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
                           "-c", str(src), "-o", str(tmp_path / "t.o")])


def test_plan_create_rejects_bad_arguments(lib):
    from paper_2512_04447_b200 import rsdft
    with pytest.raises(rsdft.RsdftError) as e:
        rsdft.rsdft_plan_create((20, 16, 16), (10.0, 10.0, 10.0))
    assert e.value.code == rsdft.RSDFT_UNSUPPORTED and "20" in str(e.value)
    with pytest.raises(rsdft.RsdftError) as e:
        rsdft.rsdft_plan_create((16, 16, 176), (10.0, 10.0, 10.0))      # 16 * 11 and not a multiple of 12
    assert e.value.code == rsdft.RSDFT_UNSUPPORTED
    with pytest.raises(rsdft.RsdftError) as e:
        rsdft.rsdft_plan_create((16, 16, 16), (10.0, -1.0, 10.0))
    assert e.value.code == rsdft.RSDFT_UNSUPPORTED
    with pytest.raises(rsdft.RsdftError) as e:
        rsdft.rsdft_plan_create((16, 0, 16), (10.0, 10.0, 10.0))
    assert e.value.code == rsdft.RSDFT_INVALID_ARG
    sp = dict(rc=2.0, l=[0, 1], m=[0, 2], D=np.eye(2), alpha=[2.0, 2.0])
    with pytest.raises(rsdft.RsdftError) as e:      # |m| > l
        rsdft.rsdft_plan_create((16, 16, 16), (10.0,) * 3, (np.zeros((1, 3)), [0]), [sp])
    assert e.value.code == rsdft.RSDFT_INVALID_ARG and "|m| > l" in str(e.value)
    sp = dict(rc=6.0, l=[0], m=[0], D=np.eye(1), alpha=[2.0])
    with pytest.raises(rsdft.RsdftError) as e:      # 2 rc >= L
        rsdft.rsdft_plan_create((16, 16, 16), (10.0,) * 3, (np.zeros((1, 3)), [0]), [sp])
    assert e.value.code == rsdft.RSDFT_UNSUPPORTED
    sp = dict(rc=2.0, l=[0, 0], m=[0, 0], D=np.array([[1.0, 0.5], [0.25, 1.0]]), alpha=[2.0, 1.0])
    with pytest.raises(rsdft.RsdftError) as e:      # D not symmetric
        rsdft.rsdft_plan_create((16, 16, 16), (10.0,) * 3, (np.zeros((1, 3)), [0]), [sp])
    assert e.value.code == rsdft.RSDFT_INVALID_ARG
    sp = dict(rc=2.0, l=[0], m=[0], D=np.eye(1), alpha=[2.0])
    with pytest.raises(rsdft.RsdftError) as e:      # species index out of range is caught on the host
        rsdft.rsdft_plan_create((16, 16, 16), (10.0,) * 3, (np.zeros((1, 3)), [3]), [sp])
    assert e.value.code in (rsdft.RSDFT_INVALID_ARG, rsdft.RSDFT_CUDA)


def test_null_plan_calls_fail_cleanly(lib):
    assert lib.rsdft_apply_h(None, 1, None, 0, None, 0, None) == -1
    assert lib.rsdft_subspace_gram(None, 1, None, 0, None, 0, None, None, 1, None) == -1
    assert lib.rsdft_plan_set_vloc(None, None, None) == -1
    assert lib.rsdft_plan_info(None, None) == -1
    assert lib.rsdft_plan_destroy(None) == 0
    assert b"null" in lib.rsdft_last_error()


def test_product_does_not_import_the_oracle():
    """The CUDA path and its binding never route through oracle/ (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2512_04447_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, re.M), f
                assert "rsdft_oracle" not in text, f
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith((".py", ".c")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+paper_2512_04447_b200", text, re.M), f
                assert "csrc" not in text.replace("paper_2512_04447_b200/csrc (the CUDA path)", ""), f
