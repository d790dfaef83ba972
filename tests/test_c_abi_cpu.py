"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/pimc.h declares,
validates arguments, and refuses to compute without a CUDA device (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1103_4887_b200 import build, binding
    build.build()
    return binding.lib()


def test_every_declared_symbol_is_exported_and_bound(L):
    import paper_1103_4887_b200 as P
    hdr = open(os.path.join(ROOT, "include", "pimc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(pimc_[a-z0-9_]+)\s*\(", hdr)))
    assert len(declared) >= 25
    for name in declared:
        assert hasattr(L, name), f"{name} declared in pimc.h but not exported by libpimc.so"
    assert sorted(P.exported_symbols()) == declared, "python binding and header disagree"


def test_shape_validation_without_touching_the_device(L):
    assert L.pimc_model_np(1, 4) == 7 and L.pimc_model_np(0, 2) == 4 and L.pimc_model_np(0, 1) == 1
    assert L.pimc_model_np(1, 3) < 0 and L.pimc_model_np(0, 5) < 0 and L.pimc_model_np(7, 2) < 0
    assert L.pimc_workspace_bytes(1, 4, 1, 32768, 1, 64) > 32769 * 4 * 8 * 6
    assert L.pimc_workspace_bytes(1, 4, 1, 32768, 1, 32) < L.pimc_workspace_bytes(1, 4, 1, 32768, 1, 64)
    assert L.pimc_workspace_bytes(1, 4, 1, 8192, 128, 64) > 128 * 8193 * 4 * 8 * 6
    for bad in ((1, 3, 1, 100, 1, 64), (0, 5, 1, 100, 1, 64), (1, 4, 5, 100, 1, 64), (1, 4, 1, 0, 1, 64), (1, 4, 1, 100, 0, 64),
                (1, 4, 1, 100, 1, 16), (9, 4, 1, 100, 1, 64)):
        assert L.pimc_workspace_bytes(*bad) == 0, bad


def test_init_rejects_bad_arguments_and_has_no_cpu_fallback(L):
    import torch
    h = C.c_void_p()
    rf = (C.c_double * 4)(100.0, 1e4, 1e4, 1e4)
    p0 = (C.c_double * 7)(120, 36, 0.3, 50, -77, -54.4, 1)
    fake_ws = C.c_void_p(256 * 1000)
    big = 1 << 30
    assert L.pimc_init(None, 1, 4, 1, 100, 0.02, 1.0, rf, p0, 1, 64, fake_ws, big, None) == -1
    assert L.pimc_init(C.byref(h), 1, 4, 1, 100, float("nan"), 1.0, rf, p0, 1, 64, fake_ws, big, None) == -1
    assert L.pimc_init(C.byref(h), 1, 4, 1, 100, 0.02, 1.0, None, p0, 1, 64, fake_ws, big, None) == -1
    assert L.pimc_init(C.byref(h), 1, 3, 1, 100, 0.02, 1.0, rf, p0, 1, 64, fake_ws, big, None) == -4
    assert L.pimc_init(C.byref(h), 1, 4, 1, 100, 0.02, 1.0, rf, p0, 1, 64, C.c_void_p(256 * 1000 + 8), big, None) == -1
    assert L.pimc_init(C.byref(h), 1, 4, 1, 100, 0.02, 1.0, rf, p0, 1, 64, fake_ws, 1000, None) == -1
    assert b"workspace" in L.pimc_last_error(None)
    badrf = (C.c_double * 4)(100.0, -1.0, 1e4, 1e4)
    assert L.pimc_init(C.byref(h), 1, 4, 1, 100, 0.02, 1.0, badrf, p0, 1, 64, fake_ws, big, None) == -1
    if not torch.cuda.is_available():
        # valid arguments, no device: must fail loudly with PIMC_ECUDA, never compute on the CPU
        assert L.pimc_init(C.byref(h), 1, 4, 1, 100, 0.02, 1.0, rf, p0, 1, 64, fake_ws, big, None) == -3
        assert b"no CPU fallback" in L.pimc_last_error(None)
        import paper_1103_4887_b200 as P
        with pytest.raises(P.PimcError):
            P.Pimc(1, 4, 1, 100, 0.02, 1.0, [100.0, 1e4, 1e4, 1e4], [120, 36, 0.3, 50, -77, -54.4, 1])
    assert L.pimc_destroy(None) == -1
    assert L.pimc_sweep(None, 1, 0) == -1


def test_product_does_not_import_the_oracle():
    # the CUDA package and the oracle share no code and neither imports the other
    pkg = os.path.join(ROOT, "paper_1103_4887_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                for needle in ("import oracle", "from oracle", "pimc_oracle", "oracle/", "oracle."):
                    assert needle not in src, f"{f} refers to the oracle ({needle!r})"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1103_4887_b200" not in src or "never imports" in src or "shares NO code" in src
            assert "import paper_1103_4887_b200" not in src and "from paper_1103_4887_b200" not in src
    wl = open(os.path.join(ROOT, "workloads", "configs.py")).read()
    assert "import oracle" not in wl and "paper_1103_4887_b200" not in wl
