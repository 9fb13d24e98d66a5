"""The C-ABI library loads and exports every symbol include/bse.h declares (no GPU needed)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bse():
    from paper_2409_15116_b200 import build
    build.build()
    from paper_2409_15116_b200 import bse as mod
    return mod


def test_header_symbols_exported(bse):
    hdr = open(os.path.join(ROOT, "include", "bse.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(bse_[a-z0-9_]+)\s*\(", hdr))
    assert {"bse_create", "bse_build_tau", "bse_apply_k1x", "bse_destroy"} <= declared
    lib = ctypes.CDLL(bse.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in bse.h but not exported"
    assert declared == set(bse.EXPORTS)


def test_no_cpu_fallback_and_argument_checks(bse):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CPU-box check")
    with pytest.raises(bse.BseError) as e:
        bse.bse_create([24] * 3, np.eye(3) * 10, 8.0, 8, np.zeros(8), 32, np.zeros(8), np.zeros(32), 0.0)
    assert e.value.code == bse.BSE_ECUDA and b"no CPU fallback" in bse.lib.bse_last_error()
    with pytest.raises(bse.BseError) as e:
        bse.bse_create([24] * 3, np.eye(3) * 10, 8.0, 8, None, 32, np.zeros(8), np.zeros(32), 0.0)
    assert e.value.code == bse.BSE_EINVAL
    with pytest.raises(bse.BseError) as e:
        bse.bse_probe_fp64_peak()
    assert e.value.code == bse.BSE_ECUDA


def test_product_path_does_not_import_oracle():
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2409_15116_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                src = open(os.path.join(root, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
