"""CPU-side checks of the boundary: libvc.so builds/loads and exports every symbol include/vc.h declares;
compute entry points fail loudly without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def v():
    from paper_1202_1350_b200 import build as vb
    vb.build()
    import paper_1202_1350_b200 as v
    v.lib()
    return v


def _declared():
    src = open(os.path.join(ROOT, "include", "vc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(vc_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(v):
    from paper_1202_1350_b200 import binding
    names = _declared()
    assert "vc_circuit_load" in names and "vc_prove_layer" in names and len(names) >= 15
    L = ctypes.CDLL(str(v.library_path()))
    for n in names:
        assert hasattr(L, n), n
    assert sorted(binding.EXPORTS) == names


def test_strerror_and_sizes(v):
    for code in range(6):
        assert v.vc_strerror(code)
    assert v.lib().vc_transcript_words(None, 0) == 0
    assert v.lib().vc_depth(None) == 0


def test_no_cpu_fallback(v):
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU-only box")
    import vc_workloads as W
    c = W.config(1)
    with pytest.raises(v.VCError) as e:
        v.vc_circuit_load(c.layers, c.log_input)
    assert e.value.code == v.VC_ERR_CUDA


def test_oracle_is_not_reachable_from_the_product():
    """The product package must not import or mention the oracle."""
    pkg = os.path.join(ROOT, "paper_1202_1350_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
