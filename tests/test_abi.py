"""The C-ABI boundary without a GPU: libcbct.so builds, loads and exports every symbol that
include/cbct.h declares; the product path holds no oracle import and fails loudly when no
sm_100 device is present (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "cbct.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cbct_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_five_north_star_calls():
    names = _declared_symbols()
    for must in ("cbct_geometry_create", "cbct_forward_project", "cbct_back_project", "cbct_tv_prox",
                 "cbct_fbs_reconstruct"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1001_0599_b200 import build, cbct
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    declared = _declared_symbols()
    assert len(declared) >= 15
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/cbct.h but not exported"
    assert sorted(cbct.EXPORTS) == declared
    assert b"sm_100a" in ctypes.cast(ctypes.CDLL(path).cbct_version, ctypes.CFUNCTYPE(ctypes.c_char_p))()


def test_library_is_built_for_sm_100a_only():
    import shutil
    import subprocess
    from paper_1001_0599_b200 import build
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", build.build()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_product_path_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_1001_0599_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), fn
                assert "cbct_oracle" not in text and "liboracle" not in text, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "csrc" not in text.replace("paper_1001_0599_b200/csrc (the CUDA", "")
            assert not re.search(r"^\s*(from|import)\s+paper_1001_0599_b200", text, flags=re.M), fn


def test_create_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1001_0599_b200 import cbct, inputs
    with pytest.raises(cbct.CbctError) as e:
        cbct.geometry_create(inputs.config(1).geom)
    assert e.value.status == 5 and "no CPU fallback" in str(e.value)


def test_argument_validation_needs_no_gpu():
    from paper_1001_0599_b200 import cbct, inputs
    g = inputs.config(1).geom
    for bad in (g.replace(nx=0), g.replace(hx=-1.0), g.replace(sad=2000.0), g.replace(bc_z=7),
                g.replace(hx=40.0, hy=40.0)):
        with pytest.raises(cbct.CbctError) as e:
            cbct.geometry_create(bad)
        assert e.value.status in (1, 2), str(e.value)
    with pytest.raises(cbct.CbctError):
        cbct.geometry_create(g.replace(nu=50), max_levels=3)     # 50 not divisible by 4
