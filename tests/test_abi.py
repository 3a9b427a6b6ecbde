"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol
include/z4c.h declares; the size queries (pure host code) agree with the documented layout; the product path
never imports the oracle and fails loudly without a GPU."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

from paper_2409_10383_b200 import build as B
from paper_2409_10383_b200 import inputs as I
from paper_2409_10383_b200 import z4c as Z

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    B.build()
    return Z.load_library()


def header_symbols():
    src = open(os.path.join(ROOT, "include", "z4c.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(z4c_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_all_exported(lib):
    syms = header_symbols()
    assert sorted(Z.SYMBOLS) == syms
    lib4 = Z.load_library(ng=4)            # the 4-ghost / 6th-order build exports the same ABI
    for s in syms:
        assert hasattr(lib, s), s
        assert hasattr(lib4, s), s


def test_library_is_sm100a_only():
    out = subprocess.run(["cuobjdump", "-lelf", Z.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert not re.search(r"sm_(?!100a)\d+", out)


def test_size_queries(lib):
    p = I.params_puncture(128, 32, 16.0, 2.0)
    cp = Z.make_params(p)
    assert lib.z4c_state_bytes(C.byref(cp)) == 22 * 64 * 38 ** 3 * 8          # 618 MB
    wb = lib.z4c_workspace_bytes(C.byref(cp))
    assert wb >= 2 * 22 * 64 * 32 ** 3 * 8 and wb % 256 == 0
    cp4 = Z.make_params(p)
    cp4.ng = 4
    assert lib.z4c_state_bytes(C.byref(cp4)) == 0                       # each build accepts only its own ghost count
    assert Z.load_library(ng=4).z4c_state_bytes(C.byref(cp4)) == 22 * 64 * 40 ** 3 * 8
    bad = Z.make_params(p)
    bad.ng = 2
    assert lib.z4c_state_bytes(C.byref(bad)) == 0 and lib.z4c_workspace_bytes(C.byref(bad)) == 0
    bad = Z.make_params(p)
    bad.n = 4
    assert lib.z4c_state_bytes(C.byref(bad)) == 0


def test_create_rejects_bad_arguments(lib):
    cp = Z.make_params(I.params_noise())
    h = C.c_void_p()
    assert lib.z4c_create(C.byref(cp), None, None, None, C.byref(h)) == Z.Z4C_EINVAL
    assert lib.z4c_create(C.byref(cp), 256, 8, None, C.byref(h)) == Z.Z4C_EINVAL      # misaligned workspace
    assert lib.z4c_step(None, 1) == Z.Z4C_EINVAL
    assert lib.z4c_last_error(None) == b"null context"


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2409_10383_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("CPU oracle", "").replace("the oracle", "").lower() \
                    or f in ("inputs.py",), f
    code = "import paper_2409_10383_b200.z4c, paper_2409_10383_b200.inputs, sys; " \
           "assert not any(m.startswith('oracle') for m in sys.modules)"
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        Z.Z4c(I.params_noise())
