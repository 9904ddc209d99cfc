"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/tqp.h declares;
host-side argument logic that needs no GPU.  (No compute calls here.)"""
import ctypes
import os
import re

import pytest

import paper_2606_07404_b200 as tq
from paper_2606_07404_b200 import binding, build


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    assert os.path.exists(path)
    lib = tq.load_library()
    declared = tq.abi_symbols()
    assert len(declared) >= 19
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/tqp.h but not exported"
    for must in ("tqp_route", "tqp_dispatch", "tqp_expert_fwd", "tqp_expert_bwd", "tqp_combine", "tqp_step_host"):
        assert must in declared


def test_header_is_plain_c_abi():
    text = open(binding.HEADER).read()
    assert 'extern "C"' in text
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)     # signatures only, comments stripped
    assert "torch" not in text.lower() and "at::" not in text and "std::" not in text


def test_workspace_bytes_and_shape_validation():
    big = tq.workspace_bytes(16384, 2560, 1024, 460, 12, 32)
    small = tq.workspace_bytes(64, 128, 256, 8, 2, 8)
    assert 0 < small < big < 180e9
    assert tq.workspace_bytes(64, 100, 256, 8, 2, 8) == 0       # d % 128 != 0 -> invalid desc
    assert tq.workspace_bytes(64, 128, 256, 8, 9, 8) == 0       # k > E
    assert tq.workspace_bytes(64, 128, 256, 8, 2, 5) == 0       # r not in {8,16,32}


def test_status_strings_and_null_handling():
    lib = tq.load_library()
    assert lib.tqp_status_string(0) == b"TQP_OK"
    assert lib.tqp_status_string(6) == b"TQP_ERR_ARCH"
    assert lib.tqp_create(None, None) == 1                         # TQP_ERR_ARG, no crash
    ctx = ctypes.c_void_p()
    bad = binding.LayerDesc(64, 100, 256, 8, 2, 8, 8, 256, 1.0, 1)
    assert lib.tqp_create(ctypes.byref(ctx), ctypes.byref(bad)) == 2   # TQP_ERR_SHAPE before touching the device
    lib.tqp_destroy(None)


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(tq.TqpError):
        tq.TqpLayer(64, 128, 256, 8, 2, 8)


def test_product_path_does_not_touch_the_oracle():
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    pkg = os.path.join(root, "paper_2606_07404_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                code = "\n".join(l for l in text.splitlines() if not l.strip().startswith(("//", "#", "*", "/*")))
                assert not re.search(r"^\s*(import|from)\s+oracle", code, flags=re.M), f
                assert "libtqp_oracle" not in code and "tqp_oracle_" not in code, f
