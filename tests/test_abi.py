"""CPU-side checks of the boundary: libkx.so builds, loads and exports every symbol include/kx.h declares;
the product path fails loudly without a GPU (no CPU fallback) and never imports oracle/."""
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "kx.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(kx_[a-z_]+)\s*\(", src)
    return sorted(set(names))


def test_header_symbols_are_exported():
    import paper_2607_00755_b200 as kx
    kx.build_library()
    declared = _declared()
    assert len(declared) >= 14 and "kx_build" in declared and "kx_evolve" in declared
    exported = kx.exported_symbols()
    assert sorted(exported) == declared
    # and nm agrees (extern "C", unmangled)
    out = subprocess.run(["nm", "-D", "--defined-only", kx.library_path()], capture_output=True, text=True).stdout
    for name in declared:
        assert re.search(rf"\bT {name}\b", out), name


def test_version_call_needs_no_gpu():
    import ctypes
    import paper_2607_00755_b200 as kx
    lib = ctypes.CDLL(kx.build_library())
    lib.kx_version.restype = ctypes.c_int32
    assert lib.kx_version() >= 100


def test_library_is_sm100a_only():
    import paper_2607_00755_b200 as kx
    out = subprocess.run(["cuobjdump", "-lelf", kx.build_library()], capture_output=True, text=True).stdout
    assert "sm_100a" in out and "sm_90" not in out and "sm_80" not in out


def test_no_cpu_fallback_without_gpu():
    import numpy as np
    import torch
    import paper_2607_00755_b200 as kx
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    p = np.linspace(0.1, 5.0, 16)
    with pytest.raises(kx.KxError):
        kx.Handle(p, np.full(16, 0.3))


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2607_00755_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "okx_" not in txt, fn
    # and the oracle never imports the product
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_2607_00755_b200 import" not in txt and "import paper_2607" not in txt and "libkx" not in txt
    code = "import sys; import paper_2607_00755_b200; assert 'oracle' not in sys.modules"
    subprocess.check_call([sys.executable, "-c", code], cwd=ROOT)
