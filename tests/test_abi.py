"""The C-ABI library loads and exports every symbol include/dft.h declares; calls that need no
device behave as documented (no CPU fallback: without a GPU, plan creation fails loudly)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2507_08578_b200 as dft

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "dft.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dft_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported():
    L = dft.lib()
    names = _declared()
    assert len(names) >= 12
    for n in names:
        assert hasattr(L, n), "libdftb200.so does not export %s" % n
    assert sorted(dft.SYMBOLS) == names


def test_argument_errors_need_no_device():
    L = dft.lib()
    out = C.c_void_p()
    rc = L.dft_plan_create(C.byref(out), None, 1, None, 1.0, None, 0, None, None, 0, None, None)
    assert rc == dft.DFT_ERR_INVALID_ARG and b"null" in L.dft_last_error()
    assert L.dft_apply_h(None, None, None, 1, None) == dft.DFT_ERR_INVALID_ARG
    assert L.dft_plan_destroy(None) == dft.DFT_OK


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    import synth
    cfg = synth.make_config("c0", with_vloc=False)
    with pytest.raises(dft.DftError) as ei:
        dft.Plan(cfg)
    assert ei.value.code == dft.DFT_ERR_CUDA


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2507_08578_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dp, f)).read()
                assert "import oracle" not in src and "oracle/" not in src.replace("oracle/ (the CPU checker)", "")
