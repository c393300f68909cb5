"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol include/dh.h declares.
(No compute calls here: those are the `-m gpu` parity tests.)"""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "dh.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dh_[a-z_]+)\s*\(", src)))


def test_header_declares_the_five_calls_of_the_boundary():
    names = _declared()
    for must in ("dh_create", "dh_cfl_dt", "dh_step", "dh_step_vjp", "dh_destroy"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2512_13403_b200 import build, dh
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for name in _declared():
        assert hasattr(lib, name), name
    assert sorted(dh.SYMBOLS) == _declared()
    lib.dh_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.dh_version()


def test_library_contains_sm100a_code_only():
    from paper_2512_13403_b200 import build
    path = build.build()
    out = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_binding_fails_loudly_without_a_gpu():
    import torch
    from paper_2512_13403_b200 import dh
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        dh.Solver(16, 16, 16)
    # the raw C call reports a CUDA error instead of silently doing anything on the CPU
    with pytest.raises(dh.DhError):
        dh.dh_create(16, 16, 16, 1.4, dh.DH_F32)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2512_13403_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "dh_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".hpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2512_13403_b200" not in txt and "from paper_2512_13403_b200" not in txt, f
            assert "csrc" not in txt and "dh_math" not in txt, f
