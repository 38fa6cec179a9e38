"""Host-side checks that need no GPU: liblam.so builds for sm_100a, loads, and exports every symbol that
include/lam.h declares; argument validation; and no CPU fallback (compute entry points fail loudly)."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_2401_11101_b200 import lam

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "lam.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lam_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_all_exported():
    lam.build()
    L = C.CDLL(lam.LIB_PATH)
    syms = declared_symbols()
    assert len(syms) >= 11
    for s in syms:
        assert hasattr(L, s), f"{s} declared in include/lam.h but not exported"
    assert sorted(lam.EXPORTS) == syms


def test_binding_has_the_same_names():
    for s in declared_symbols():
        assert callable(getattr(lam, s)), s


def test_default_params_match_header_comment():
    p = lam.lam_default_params()
    assert (p.kernel, p.width, p.filter, p.input) == (0, 6, 1, 0)
    assert p.oversample == 2.0 and p.center_u != p.center_u  # NaN


def test_validation_happens_before_any_device_use():
    with pytest.raises(lam.LamError) as e:
        lam.lam_create(63, 64, 64, [0.0], 0.3)
    assert e.value.status == lam.LAM_EINVAL and "even" in str(e.value)
    with pytest.raises(lam.LamError) as e:
        lam.lam_create(48, 64, 64, [0.0], 0.3)
    assert e.value.status == lam.LAM_EUNSUPPORTED


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback_without_a_device():
    with pytest.raises(lam.LamError) as e:
        lam.lam_create(64, 64, 64, [0.0, 1.0], 0.3)
    assert e.value.status == lam.LAM_ECUDA


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2401_11101_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert "oracle" not in open(os.path.join(dp, f)).read().replace("oracle/", "").replace(
                    "the oracle", "").replace("oracle-side", ""), f
